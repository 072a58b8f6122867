// precond.cu -- block-diagonal preconditioner: celes_partition, celes_precond_setup,
// celes_precond_apply.  Kernels in precond_kernels.cuh; the LU factorisation of the blocks is cuSOLVER's getrf / getrs.
#include <cuda_runtime.h>
#include <cusolverDn.h>

#include <algorithm>
#include <chrono>
#include <cmath>
#include <cstring>
#include <vector>

#include "ctx.h"
#include "partition.h"
#include "precond_kernels.cuh"
#include "translation_table.h"

void celes::host::free_precond(celes_ctx* c) {
    cudaFree(c->pc_order); cudaFree(c->pc_grp_offset); cudaFree(c->pc_blk_offset); cudaFree(c->pc_cta_group);
    cudaFree(c->pc_cta_row0); cudaFree(c->pc_blocks); cudaFree(c->pc_tmp);
    c->pc_order = c->pc_grp_offset = c->pc_cta_group = c->pc_cta_row0 = nullptr;
    c->pc_blk_offset = nullptr; c->pc_blocks = c->pc_tmp = nullptr;
    c->pc_ready = false; c->pc_groups = c->pc_max_n = c->pc_ctas = 0; c->pc_elems = 0;
}

// z = blockdiag(M_j^{-1}) v  (step 4)
int celes::host::precond_apply(celes_ctx* c, const float2* v, float2* z, cudaStream_t s) {
    celes::block_gemv_kernel<<<c->pc_ctas, celes::kGemvRows, (size_t)c->pc_max_n * sizeof(float2), s>>>(
        c->nmax, c->pc_cta_group, c->pc_cta_row0, c->pc_grp_offset, c->pc_order, c->pc_blk_offset, c->pc_blocks, v, z);
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
// (3) LU factorisation with partial pivoting (cuSOLVER getrf), here followed by the solve against the identity
// (getrs) so that (4) applying M_j^{-1} is a batched matrix-vector product (block_gemv_kernel).
int celes_precond_setup(celes_ctx* ctx, const double* edge_xyz, celes_precond_info* info, void* cuda_stream) {
    if (!ctx || !edge_xyz) return CELES_EINVAL;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const auto t_start = std::chrono::steady_clock::now();
    free_precond(ctx);
    celes::Partition part;
    if (!celes::build_partition(ctx->N, ctx->pos.data(), edge_xyz, part)) return CELES_EINVAL;
    const int G = part.n_groups(), nmax = ctx->nmax, H = nmax / 2, P = 2 * ctx->lmax + 1;
    const long long max_n = (long long)part.max_group() * nmax;
    if (max_n * (long long)sizeof(float2) > 200 * 1024) return CELES_EINVAL;      // subset too large for one CTA's x slice
    std::vector<long long> blk_off(G), pair_off(G + 1, 0);
    std::vector<int> cta_group, cta_row0;
    long long elems = 0;
    for (int j = 0; j < G; ++j) {
        const long long nj = part.offset[j + 1] - part.offset[j], n = nj * nmax;
        blk_off[j] = elems;
        elems += n * n;
        pair_off[j + 1] = pair_off[j] + nj * nj;
        for (long long r = 0; r < n; r += celes::kGemvRows) { cta_group.push_back(j); cta_row0.push_back((int)r); }
    }
    if (pair_off[G] > 0x7fffffffLL) return CELES_EINVAL;
    std::vector<double> a5d, b5d;
    if (!celes::build_translation_table(ctx->lmax, a5d, b5d)) return CELES_EINVAL;
    std::vector<float> a5f(a5d.begin(), a5d.end()), b5f(b5d.begin(), b5d.end());

    long long* d_pair_off = nullptr;
    float *d_a5 = nullptr, *d_b5 = nullptr;
    int* d_info = nullptr;
    constexpr int kPcStreams = 8;
    struct Lane { cudaStream_t stream = nullptr; cusolverDnHandle_t handle = nullptr; float2* lu = nullptr;
                  int* ipiv = nullptr; void* work = nullptr; };
    Lane lanes[kPcStreams];
    const int nstreams = std::max(1, std::min(kPcStreams, G));
    auto cleanup = [&](int code) {
        cudaFree(d_pair_off); cudaFree(d_a5); cudaFree(d_b5); cudaFree(d_info);
        for (Lane& ln : lanes) {
            if (ln.stream) cudaStreamSynchronize(ln.stream);
            if (ln.handle) cusolverDnDestroy(ln.handle);
            cudaFree(ln.lu); cudaFree(ln.ipiv); cudaFree(ln.work);
            if (ln.stream) cudaStreamDestroy(ln.stream);
        }
        if (code != CELES_OK) free_precond(ctx);
        return code;
    };
#define PC_TRY(expr)                                                                                   \
    do {                                                                                               \
        cudaError_t e_ = (expr);                                                                       \
        if (e_ != cudaSuccess) return cleanup(e_ == cudaErrorMemoryAllocation ? CELES_ENOMEM : CELES_ECUDA); \
    } while (0)
    PC_TRY(cudaMalloc(&ctx->pc_order, sizeof(int) * ctx->N));
    PC_TRY(cudaMalloc(&ctx->pc_grp_offset, sizeof(int) * (G + 1)));
    PC_TRY(cudaMalloc(&ctx->pc_blk_offset, sizeof(long long) * G));
    PC_TRY(cudaMalloc(&ctx->pc_cta_group, sizeof(int) * cta_group.size()));
    PC_TRY(cudaMalloc(&ctx->pc_cta_row0, sizeof(int) * cta_row0.size()));
    PC_TRY(cudaMalloc(&ctx->pc_blocks, sizeof(float2) * (size_t)elems));
    PC_TRY(cudaMalloc(&ctx->pc_tmp, sizeof(float2) * (size_t)ctx->N * nmax));
    PC_TRY(cudaMalloc(&d_pair_off, sizeof(long long) * (G + 1)));
    PC_TRY(cudaMalloc(&d_a5, sizeof(float) * a5f.size()));
    PC_TRY(cudaMalloc(&d_b5, sizeof(float) * b5f.size()));
    PC_TRY(cudaMalloc(&d_info, sizeof(int) * 2 * (size_t)G));
    PC_TRY(cudaMemcpyAsync(ctx->pc_order, part.order.data(), sizeof(int) * ctx->N, cudaMemcpyHostToDevice, s));
    PC_TRY(cudaMemcpyAsync(ctx->pc_grp_offset, part.offset.data(), sizeof(int) * (G + 1), cudaMemcpyHostToDevice, s));
    PC_TRY(cudaMemcpyAsync(ctx->pc_blk_offset, blk_off.data(), sizeof(long long) * G, cudaMemcpyHostToDevice, s));
    PC_TRY(cudaMemcpyAsync(ctx->pc_cta_group, cta_group.data(), sizeof(int) * cta_group.size(), cudaMemcpyHostToDevice, s));
    PC_TRY(cudaMemcpyAsync(ctx->pc_cta_row0, cta_row0.data(), sizeof(int) * cta_row0.size(), cudaMemcpyHostToDevice, s));
    PC_TRY(cudaMemcpyAsync(d_pair_off, pair_off.data(), sizeof(long long) * (G + 1), cudaMemcpyHostToDevice, s));
    PC_TRY(cudaMemcpyAsync(d_a5, a5f.data(), sizeof(float) * a5f.size(), cudaMemcpyHostToDevice, s));
    PC_TRY(cudaMemcpyAsync(d_b5, b5f.data(), sizeof(float) * b5f.size(), cudaMemcpyHostToDevice, s));
    (void)H; (void)P;
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
    // (3) factorise and invert block by block; the blocks are independent and small against the device, so they
    // are spread round-robin over kPcStreams streams (own cuSOLVER handle and scratch each) that fork from and join s
    {
        cudaEvent_t ev_fork = nullptr;
        PC_TRY(cudaEventCreateWithFlags(&ev_fork, cudaEventDisableTiming));
        cudaEventRecord(ev_fork, s);
        int status = CELES_OK;
        for (int q = 0; q < nstreams && status == CELES_OK; ++q) {
            if (cudaStreamCreateWithFlags(&lanes[q].stream, cudaStreamNonBlocking) != cudaSuccess ||
                cusolverDnCreate(&lanes[q].handle) != CUSOLVER_STATUS_SUCCESS ||
                cusolverDnSetStream(lanes[q].handle, lanes[q].stream) != CUSOLVER_STATUS_SUCCESS) { status = CELES_ECUDA; break; }
            int lwork = 0;
            if (cudaMalloc(&lanes[q].lu, sizeof(float2) * (size_t)(max_n * max_n)) != cudaSuccess ||
                cudaMalloc(&lanes[q].ipiv, sizeof(int) * (size_t)max_n) != cudaSuccess) { status = CELES_ENOMEM; break; }
            if (cusolverDnCgetrf_bufferSize(lanes[q].handle, (int)max_n, (int)max_n, (cuComplex*)lanes[q].lu, (int)max_n,
                                            &lwork) != CUSOLVER_STATUS_SUCCESS) { status = CELES_ECUDA; break; }
            if (cudaMalloc(&lanes[q].work, sizeof(cuComplex) * (size_t)std::max(lwork, 1)) != cudaSuccess) { status = CELES_ENOMEM; break; }
            cudaStreamWaitEvent(lanes[q].stream, ev_fork, 0);
        }
        for (int j = 0; j < G && status == CELES_OK; ++j) {
            Lane& ln = lanes[j % nstreams];
            const int n = (part.offset[j + 1] - part.offset[j]) * nmax;
            float2* Mj = ctx->pc_blocks + blk_off[j];
            if (cudaMemcpyAsync(ln.lu, Mj, sizeof(float2) * (size_t)n * n, cudaMemcpyDeviceToDevice, ln.stream) != cudaSuccess) status = CELES_ECUDA;
            const int ib = (int)std::min<long long>(((long long)n * n + 255) / 256, (long long)ctx->sm_count * 8);
            celes::set_identity_kernel<<<ib, 256, 0, ln.stream>>>(n, Mj);
            if (cusolverDnCgetrf(ln.handle, n, n, (cuComplex*)ln.lu, n, (cuComplex*)ln.work, ln.ipiv, d_info + 2 * j) !=
                CUSOLVER_STATUS_SUCCESS) status = CELES_ECUDA;
            if (cusolverDnCgetrs(ln.handle, CUBLAS_OP_N, n, n, (const cuComplex*)ln.lu, n, ln.ipiv, (cuComplex*)Mj, n,
                                 d_info + 2 * j + 1) != CUSOLVER_STATUS_SUCCESS) status = CELES_ECUDA;
        }
        for (int q = 0; q < nstreams; ++q) {                   // join
            if (!lanes[q].stream) continue;
            cudaEvent_t ev = nullptr;
            if (cudaEventCreateWithFlags(&ev, cudaEventDisableTiming) == cudaSuccess) {
                cudaEventRecord(ev, lanes[q].stream);
                cudaStreamWaitEvent(s, ev, 0);
                cudaEventDestroy(ev);
            } else {
                cudaStreamSynchronize(lanes[q].stream);
            }
        }
        cudaEventDestroy(ev_fork);
        if (status != CELES_OK) { cudaStreamSynchronize(s); return cleanup(status); }
    }
    std::vector<int> infos(2 * (size_t)G);
    PC_TRY(cudaMemcpyAsync(infos.data(), d_info, sizeof(int) * infos.size(), cudaMemcpyDeviceToHost, s));
    PC_TRY(cudaStreamSynchronize(s));
#undef PC_TRY
    for (int v : infos) if (v != 0) return cleanup(CELES_ECUDA);     // singular block or bad argument
    ctx->pc_groups = G; ctx->pc_max_n = (int)max_n; ctx->pc_ctas = (int)cta_group.size(); ctx->pc_elems = elems;
    ctx->pc_ready = true;
    cudaFuncSetAttribute(celes::block_gemv_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(max_n * sizeof(float2)));
    if (info) {
        info->n_groups = G;
        info->max_group_spheres = part.max_group();
        info->block_bytes = elems * (long long)sizeof(float2);
        info->seconds = std::chrono::duration<double>(std::chrono::steady_clock::now() - t_start).count();
    }
    return cleanup(CELES_OK);
}

int celes_precond_apply(celes_ctx* ctx, const void* v_dev, void* z_dev, void* cuda_stream) {
    if (!ctx || !v_dev || !z_dev || v_dev == z_dev || !ctx->pc_ready) return CELES_EINVAL;
    return precond_apply(ctx, (const float2*)v_dev, (float2*)z_dev, (cudaStream_t)cuda_stream);
}

}  // extern "C"
