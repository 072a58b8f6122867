// precond.cu -- block-diagonal preconditioner: celes_partition, celes_precond_setup,
// celes_precond_apply.  Kernels in precond_kernels.cuh (assembly, apply) and block_inverse.cuh (pivoted elimination).
#include <cuda_runtime.h>

#include <algorithm>
#include <chrono>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <vector>

#include "ctx.h"
#include "block_inverse.cuh"
#include "partition.h"
#include "precond_kernels.cuh"
#include "translation_table.h"

// the preconditioner's arrays are pieces of pc_arena; pc_blocks is its own allocation
static void forget_precond(celes_ctx* c) {
    c->pc_order = c->pc_grp_offset = c->pc_cta_group = c->pc_cta_row0 = c->pc_perm = nullptr;
    c->pc_blk_offset = nullptr; c->pc_tmp = nullptr;
    c->pc_ready = false; c->pc_groups = c->pc_max_n = c->pc_ctas = 0; c->pc_elems = 0;
}

void celes::host::free_precond(celes_ctx* c) {
    cudaFree(c->pc_arena); cudaFree(c->pc_blocks);
    c->pc_arena = nullptr; c->pc_arena_bytes = 0; c->pc_blocks = nullptr; c->pc_capacity = 0;
    forget_precond(c);
}

// z = blockdiag(M_j^{-1}) v  (step 4)
int celes::host::precond_apply(celes_ctx* c, const float2* v, float2* z, cudaStream_t s) {
    if (c->pc_max_n > celes::kGemvChunkedFrom) {               // tall blocks: x streamed through a fixed chunk of shared memory
        celes::block_gemv_chunked_kernel<<<c->pc_ctas, celes::kGemvRows, 0, s>>>(
            c->nmax, c->pc_cta_group, c->pc_cta_row0, c->pc_grp_offset, c->pc_order, c->pc_blk_offset, c->pc_perm, c->pc_blocks, v, z);
        return cudaGetLastError() == cudaSuccess ? CELES_OK : CELES_ECUDA;
    }
    const size_t smem = (size_t)c->pc_max_n * sizeof(float2);
    if (smem > 48 * 1024) {
        // the attribute belongs to the kernel, not to a context: raise it to the device limit (never lower it) and
        // leave the per-launch size to the launch
        static int optin_set = 0;
        if (!optin_set) {
            int optin = 0;
            CU_TRY(cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, c->device));
            CU_TRY(cudaFuncSetAttribute(celes::block_gemv_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, optin));
            optin_set = 1;
        }
    }
    celes::block_gemv_kernel<<<c->pc_ctas, celes::kGemvRows, smem, s>>>(
        c->nmax, c->pc_cta_group, c->pc_cta_row0, c->pc_grp_offset, c->pc_order, c->pc_blk_offset, c->pc_perm, c->pc_blocks, v, z);
    return cudaGetLastError() == cudaSuccess ? CELES_OK : CELES_ECUDA;
}

using celes::host::free_precond;
using celes::host::precond_apply;

extern "C" {

static int partition_impl(int N, const double* pos_xyz, const double* edge_xyz, int* group_of, int* n_groups) {
    if (N < 1 || !pos_xyz || !edge_xyz || !group_of) return CELES_EINVAL;
    celes::Partition part;
    if (!celes::build_partition(N, pos_xyz, edge_xyz, part)) return CELES_EINVAL;
    std::memcpy(group_of, part.group_of.data(), sizeof(int) * (size_t)N);
    if (n_groups) *n_groups = part.n_groups();
    return CELES_OK;
}

int celes_partition(int N, const double* pos_xyz, const double* edge_xyz, int* group_of, int* n_groups) {
    CELES_NOTHROW(partition_impl(N, pos_xyz, edge_xyz, group_of, n_groups))
}

// Block-diagonal preconditioner: (1) cuboid partition, (2) blocks M_j = 1 - T W on the device,
// (3) elimination with partial (row) pivoting of every block, here carried through to the explicit inverse
// (block_inverse.cuh: blocked in-place Gauss-Jordan, all blocks in the same launches) so that (4) applying M_j^{-1} is a
// batched matrix-vector product (block_gemv_kernel).
static int precond_setup_impl(celes_ctx* ctx, const double* edge_xyz, celes_precond_info* info, cudaStream_t s) {
    const auto t_start = std::chrono::steady_clock::now();
    const bool dbg = std::getenv("CELES_DEBUG") != nullptr;
    auto since = [&]() { return std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t_start).count(); };
    double t_free0 = 0, t_part = 0, t_tables = 0, t_alloc = 0, t_h2d = 0, t_gpu = 0;
    // a set-up that replaces an earlier one keeps the block buffer and the arena if the new preconditioner fits: it then
    // calls no allocator at all (cudaMalloc / cudaFree were measured at 1 ms ... 140 ms per set-up, unpredictably)
    if (ctx->pc_ready && cudaDeviceSynchronize() != cudaSuccess) return CELES_ECUDA;   // nothing may still read the arrays about to be rewritten
    forget_precond(ctx);
    t_free0 = since();
    celes::Partition part;
    if (!celes::build_partition(ctx->N, ctx->pos.data(), edge_xyz, part)) return CELES_EINVAL;
    const int G = part.n_groups(), nmax = ctx->nmax;
    t_part = since();
    const long long max_n = (long long)part.max_group() * nmax;
    if (max_n * (long long)sizeof(float2) > 200 * 1024) return CELES_EINVAL;      // subset too large for one CTA's x slice
    std::vector<long long> blk_off(G), pair_off(G + 1, 0);
    std::vector<int> cta_group, cta_row0, rounds(G), by_size(G);
    long long elems = 0;
    for (int j = 0; j < G; ++j) {
        const long long nj = part.offset[j + 1] - part.offset[j], n = nj * nmax;
        blk_off[j] = elems;
        elems += n * n;
        pair_off[j + 1] = pair_off[j] + nj * nj;
        rounds[j] = (int)((n + celes::kGjNb - 1) / celes::kGjNb);
        by_size[j] = j;
        for (long long r = 0; r < n; r += celes::kGemvRows) { cta_group.push_back(j); cta_row0.push_back((int)r); }
    }
    if (pair_off[G] > 0x7fffffffLL) return CELES_EINVAL;
    // the blocks still being eliminated in a round are a prefix of the blocks ordered by size
    std::stable_sort(by_size.begin(), by_size.end(), [&](int a, int b) { return rounds[a] > rounds[b]; });
    std::vector<long long> tile_off(G + 1, 0);
    for (int q = 0; q < G; ++q) {
        const long long n = (long long)(part.offset[by_size[q] + 1] - part.offset[by_size[q]]) * nmax;
        const long long td = (n + celes::kGjTile - 1) / celes::kGjTile;
        tile_off[q + 1] = tile_off[q] + td;
    }
    if (tile_off[G] > 0x7fffffffLL) return CELES_EINVAL;
    std::vector<double> a5d, b5d;
    if (!celes::build_translation_table(ctx->lmax, a5d, b5d)) return CELES_EINVAL;
    std::vector<float> a5f(a5d.begin(), a5d.end()), b5f(b5d.begin(), b5d.end());
    t_tables = since();

    long long *d_pair_off = nullptr, *d_tile_off = nullptr;
    float *d_a5 = nullptr, *d_b5 = nullptr;
    int *d_info = nullptr, *d_by_size = nullptr, *d_src_row = nullptr, *d_disp_count = nullptr, *d_disp_rows = nullptr;
    auto cleanup = [&](int code) {
        if (code != CELES_OK) free_precond(ctx);
        return code;
    };
#define PC_TRY(expr)                                                                                   \
    do {                                                                                               \
        cudaError_t e_ = (expr);                                                                       \
        if (e_ != cudaSuccess) {                                                                       \
            if (std::getenv("CELES_DEBUG")) std::fprintf(stderr, "celes_precond_setup: %s at line %d\n", cudaGetErrorString(e_), __LINE__); \
            return cleanup(e_ == cudaErrorMemoryAllocation ? CELES_ENOMEM : CELES_ECUDA);               \
        }                                                                                              \
    } while (0)
    const size_t rows = (size_t)ctx->N * nmax;
    // every array but the blocks is a 256-byte aligned piece of one arena (persistent tables first, temporaries after)
    size_t arena_need = 0;
    auto piece = [&](size_t bytes) { const size_t at = arena_need; arena_need += (bytes + 255) & ~(size_t)255; return at; };
    const size_t o_order = piece(sizeof(int) * ctx->N), o_grp = piece(sizeof(int) * (G + 1)), o_blk = piece(sizeof(long long) * G),
                 o_ctag = piece(sizeof(int) * cta_group.size()), o_ctar = piece(sizeof(int) * cta_row0.size()),
                 o_perm = piece(sizeof(int) * rows), o_tmp = piece(sizeof(float2) * rows), o_src = piece(sizeof(int) * rows),
                 o_pair = piece(sizeof(long long) * (G + 1)), o_tile = piece(sizeof(long long) * (G + 1)),
                 o_a5 = piece(sizeof(float) * a5f.size()), o_b5 = piece(sizeof(float) * b5f.size()), o_info = piece(sizeof(int) * (size_t)G),
                 o_dc = piece(sizeof(int) * (size_t)G), o_dr = piece(sizeof(int) * (size_t)G * celes::kGjNb), o_bs = piece(sizeof(int) * (size_t)G);
    if (ctx->pc_arena_bytes < arena_need) {
        cudaFree(ctx->pc_arena);
        ctx->pc_arena = nullptr; ctx->pc_arena_bytes = 0;
        PC_TRY(cudaMalloc(&ctx->pc_arena, arena_need));
        ctx->pc_arena_bytes = arena_need;
    }
    if (ctx->pc_capacity < elems) {
        cudaFree(ctx->pc_blocks);
        ctx->pc_blocks = nullptr; ctx->pc_capacity = 0;
        PC_TRY(cudaMalloc(&ctx->pc_blocks, sizeof(float2) * (size_t)elems));
        ctx->pc_capacity = elems;
    }
    char* A = ctx->pc_arena;
    ctx->pc_order = (int*)(A + o_order); ctx->pc_grp_offset = (int*)(A + o_grp); ctx->pc_blk_offset = (long long*)(A + o_blk);
    ctx->pc_cta_group = (int*)(A + o_ctag); ctx->pc_cta_row0 = (int*)(A + o_ctar); ctx->pc_perm = (int*)(A + o_perm);
    ctx->pc_tmp = (float2*)(A + o_tmp); d_src_row = (int*)(A + o_src); d_pair_off = (long long*)(A + o_pair);
    d_tile_off = (long long*)(A + o_tile); d_a5 = (float*)(A + o_a5); d_b5 = (float*)(A + o_b5); d_info = (int*)(A + o_info);
    d_disp_count = (int*)(A + o_dc); d_disp_rows = (int*)(A + o_dr); d_by_size = (int*)(A + o_bs);
    t_alloc = since();
    PC_TRY(cudaMemcpyAsync(ctx->pc_order, part.order.data(), sizeof(int) * ctx->N, cudaMemcpyHostToDevice, s));
    PC_TRY(cudaMemcpyAsync(ctx->pc_grp_offset, part.offset.data(), sizeof(int) * (G + 1), cudaMemcpyHostToDevice, s));
    PC_TRY(cudaMemcpyAsync(ctx->pc_blk_offset, blk_off.data(), sizeof(long long) * G, cudaMemcpyHostToDevice, s));
    PC_TRY(cudaMemcpyAsync(ctx->pc_cta_group, cta_group.data(), sizeof(int) * cta_group.size(), cudaMemcpyHostToDevice, s));
    PC_TRY(cudaMemcpyAsync(ctx->pc_cta_row0, cta_row0.data(), sizeof(int) * cta_row0.size(), cudaMemcpyHostToDevice, s));
    PC_TRY(cudaMemcpyAsync(d_pair_off, pair_off.data(), sizeof(long long) * (G + 1), cudaMemcpyHostToDevice, s));
    PC_TRY(cudaMemcpyAsync(d_tile_off, tile_off.data(), sizeof(long long) * (G + 1), cudaMemcpyHostToDevice, s));
    PC_TRY(cudaMemcpyAsync(d_a5, a5f.data(), sizeof(float) * a5f.size(), cudaMemcpyHostToDevice, s));
    PC_TRY(cudaMemcpyAsync(d_b5, b5f.data(), sizeof(float) * b5f.size(), cudaMemcpyHostToDevice, s));
    PC_TRY(cudaMemcpyAsync(d_by_size, by_size.data(), sizeof(int) * (size_t)G, cudaMemcpyHostToDevice, s));
    PC_TRY(cudaMemsetAsync(d_info, 0, sizeof(int) * (size_t)G, s));
    t_h2d = since();
    // (2) assemble every block
    {
        const unsigned grid = (unsigned)pair_off[G];
#define PC_ASM(L)                                                                                              \
    celes::assemble_blocks_kernel<L><<<grid, celes::kAsmThreads, 0, s>>>(G, d_pair_off, ctx->pc_grp_offset,     \
        ctx->pc_order, ctx->pc_blk_offset, ctx->kpos, ctx->tdiag, d_a5, d_b5, ctx->pc_blocks)
        switch (ctx->lmax) {
            case 1: PC_ASM(1); break;
            case 2: PC_ASM(2); break;
            case 3: PC_ASM(3); break;
            case 4: PC_ASM(4); break;
            case 5: PC_ASM(5); break;
            default: return cleanup(CELES_EINVAL);
        }
#undef PC_ASM
        PC_TRY(cudaGetLastError());
    }
    // (3) eliminate: one panel launch + one update launch per round of 32 columns, every block that still has columns
    {
        int optin = 0;
        PC_TRY(cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, ctx->device));
        optin -= 1024;                                                              // the kernel's static shared memory
        PC_TRY(cudaFuncSetAttribute(celes::gj_panel_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, optin));
        const int src_capacity = (int)((max_n + 3) / 4 * 4);                        // ints, keeps the panel 16-byte aligned
        const long long room = ((long long)optin - (long long)src_capacity * (long long)sizeof(int)) / (long long)sizeof(float2);
        const long long panel_capacity = std::max(0LL, std::min(room, max_n * celes::kGjNb));   // elements; larger panels work in global memory
        const size_t smem = (size_t)src_capacity * sizeof(int) + (size_t)panel_capacity * sizeof(float2);
        celes::GjBlocks B{nmax, d_by_size, ctx->pc_grp_offset, ctx->pc_blk_offset, ctx->pc_blocks, d_src_row, d_disp_count,
                          d_disp_rows, ctx->pc_perm, d_info};
        const int max_rounds = rounds[by_size[0]];
        int n_active = G;
        for (int r = 0; r < max_rounds; ++r) {
            while (n_active > 0 && rounds[by_size[n_active - 1]] <= r) --n_active;
            celes::gj_panel_kernel<<<n_active, celes::kGjThreads, smem, s>>>(B, r, src_capacity, panel_capacity);
            celes::gj_update_kernel<<<(unsigned)tile_off[n_active], 256, 0, s>>>(B, r, n_active, d_tile_off);
        }
        PC_TRY(cudaGetLastError());
    }
    std::vector<int> infos((size_t)G);
    PC_TRY(cudaMemcpyAsync(infos.data(), d_info, sizeof(int) * infos.size(), cudaMemcpyDeviceToHost, s));
    PC_TRY(cudaStreamSynchronize(s));
    t_gpu = since();
#undef PC_TRY
    for (int v : infos)
        if (v != 0) {                                                // singular block
            if (std::getenv("CELES_DEBUG")) std::fprintf(stderr, "celes_precond_setup: singular block\n");
            return cleanup(CELES_ECUDA);
        }
    ctx->pc_groups = G; ctx->pc_max_n = (int)max_n; ctx->pc_ctas = (int)cta_group.size(); ctx->pc_elems = elems;
    ctx->pc_ready = true;
    if (info) {
        info->n_groups = G;
        info->max_group_spheres = part.max_group();
        info->block_bytes = elems * (long long)sizeof(float2);
        info->seconds = std::chrono::duration<double>(std::chrono::steady_clock::now() - t_start).count();
    }
    const int rc_done = cleanup(CELES_OK);
    if (dbg)
        std::fprintf(stderr, "celes_precond_setup ms: free-old %.2f | partition %.2f | tables %.2f | alloc %.2f | h2d %.2f | gpu %.2f | free-tmp %.2f (cumulative)\n",
                     t_free0, t_part, t_tables, t_alloc, t_h2d, t_gpu, since());
    return rc_done;
}

int celes_precond_setup(celes_ctx* ctx, const double* edge_xyz, celes_precond_info* info, void* cuda_stream) {
    if (!ctx || !edge_xyz) return CELES_EINVAL;
    CELES_NOTHROW(precond_setup_impl(ctx, edge_xyz, info, (cudaStream_t)cuda_stream))
}

int celes_precond_apply(celes_ctx* ctx, const void* v_dev, void* z_dev, void* cuda_stream) {
    if (!ctx || !v_dev || !z_dev || v_dev == z_dev || !ctx->pc_ready) return CELES_EINVAL;
    return precond_apply(ctx, (const float2*)v_dev, (float2*)z_dev, (cudaStream_t)cuda_stream);
}

}  // extern "C"
