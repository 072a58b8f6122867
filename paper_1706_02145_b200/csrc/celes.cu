// celes.cu -- C-ABI library of the B200-native CELES hot path (include/celes.h).
//
// Host side of the boundary: argument validation, context (device tables + work space), kernel launches for
// y = W b (eq. 6-7) and out = b - T (W b) (eq. 8-9), and the host-driven
// restarted GMRES of celes_solve whose vector work is device kernels (krylov_kernels.cuh).
// Nothing here falls back to the CPU: without a device every compute entry point returns CELES_ECUDA.
#include <cuda_runtime.h>

#include <algorithm>
#include <chrono>
#include <cmath>
#include <complex>
#include <cstdint>
#include <cstring>
#include <functional>
#include <new>
#include <vector>

#include "../../include/celes.h"
#include "coupling_kernel.cuh"
#include "far_field.cuh"
#include "gaussian_beam.cuh"
#include "krylov_kernels.cuh"
#include "near_field.cuh"
#include "partition.h"
#include "precond_kernels.cuh"
#include "translation_table.h"

#include <cusolverDn.h>

struct celes_ctx {
    int N = 0, lmax = 0, nmax = 0;
    double k = 0.0;
    int device = 0, sm_count = 0;
    int rblocks = 0, splits = 1, chunk = 0, etile = 32;
    int variant = celes::kRotated;   // CELES_TRANSLATION_*: packed rotated (default), direct sum, scalar rotated
    size_t coupling_smem = 0;
    std::vector<double> pos;     // host copy of the centres [N][3] (partition of the preconditioner)
    double* kpos = nullptr;      // [N][3] FP64, k * r_i
    float2* tdiag = nullptr;     // [N][nmax] T diagonal Q^i_{tau,l} expanded over m (B.1)
    float4* htab = nullptr;      // Hankel lookup table [nodes][2 lmax + 1] (CELES_HANKEL_TABLE), else null
    HankelTable htab_desc = {nullptr, 0.0f, 0.0f, 0};
    float2* bpm = nullptr;       // [N][nmax] work: [b_+ | b_-]
    float2* ypart = nullptr;     // [splits][N][nmax] work: partial sums of the emitter splits
    float2 *host_in = nullptr, *host_out = nullptr;   // [N][nmax] staging of the *_host entry points (allocated on first use)
    // Krylov work space (allocated on the first celes_solve)
    int kry_restart = 0, dot_blocks = 0;
    float2* V = nullptr;         // [restart+1][n] basis
    float2* rhs = nullptr;       // [n] T a_in
    float2* tmp = nullptr;       // [n]
    double2* partial = nullptr;  // [dot_blocks][restart+1]
    double2* coef = nullptr;     // [restart+2]
    double2* hsum = nullptr;     // [2][restart+2]
    double2* hhost = nullptr;    // pinned [3][restart+2]: two Hessenberg-column halves + coefficient upload
    cudaEvent_t kry_ev[2] = {nullptr, nullptr};   // 'Hessenberg column copied' events of the look-ahead Arnoldi loop
    // block-diagonal preconditioner (celes_precond_setup)
    bool pc_ready = false;
    int pc_groups = 0, pc_max_n = 0, pc_ctas = 0;
    long long pc_elems = 0;      // sum_j n_j^2
    int* pc_order = nullptr;     // [N]
    int* pc_grp_offset = nullptr;        // [groups+1]
    long long* pc_blk_offset = nullptr;  // [groups]
    int* pc_cta_group = nullptr;         // [pc_ctas]
    int* pc_cta_row0 = nullptr;          // [pc_ctas]
    float2* pc_blocks = nullptr;         // explicit inverses M_j^{-1}, column-major, back to back
    float2* pc_tmp = nullptr;            // [n] work vector of the preconditioned solve
};

namespace {

using celes::kBlock;

#define CU_TRY(expr)                                  \
    do {                                              \
        cudaError_t e_ = (expr);                      \
        if (e_ != cudaSuccess) {                      \
            return e_ == cudaErrorMemoryAllocation ? CELES_ENOMEM : CELES_ECUDA; \
        }                                             \
    } while (0)

template <int LMAX, int ROT, bool TAB>
int launch_coupling_tt(const celes_ctx* c, cudaStream_t s) {
    const size_t smem = celes::coupling_smem_bytes<LMAX>(c->etile);
    dim3 grid(c->rblocks, c->splits);
    celes::coupling_kernel<LMAX, ROT, TAB><<<grid, kBlock, smem, s>>>(c->N, c->chunk, c->etile, c->htab_desc, c->kpos,
                                                                      c->bpm, c->ypart);
    return cudaGetLastError() == cudaSuccess ? CELES_OK : CELES_ECUDA;
}

template <int LMAX, int ROT, bool TAB>
int prepare_coupling_tt(celes_ctx* c, int* ctas_per_sm) {
    const size_t smem = celes::coupling_smem_bytes<LMAX>(c->etile);
    c->coupling_smem = smem;
    CU_TRY(cudaFuncSetAttribute(celes::coupling_kernel<LMAX, ROT, TAB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    CU_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(ctas_per_sm, celes::coupling_kernel<LMAX, ROT, TAB>, kBlock, smem));
    return CELES_OK;
}

// the table look-up exists for the default (packed rotated) body only
template <int LMAX, int ROT>
int launch_coupling_t(const celes_ctx* c, cudaStream_t s) {
    if constexpr (ROT == celes::kRotated) { if (c->htab) return launch_coupling_tt<LMAX, ROT, true>(c, s); }
    return launch_coupling_tt<LMAX, ROT, false>(c, s);
}

template <int LMAX, int ROT>
int prepare_coupling_t(celes_ctx* c, int* ctas_per_sm) {
    if constexpr (ROT == celes::kRotated) { if (c->htab) return prepare_coupling_tt<LMAX, ROT, true>(c, ctas_per_sm); }
    return prepare_coupling_tt<LMAX, ROT, false>(c, ctas_per_sm);
}

#define CELES_DISPATCH(fn, ...)                                                                              \
    switch (c->lmax * 3 + c->variant) {                                                                      \
        case 3: return fn<1, 0>(__VA_ARGS__); case 4: return fn<1, 1>(__VA_ARGS__); case 5: return fn<1, 2>(__VA_ARGS__);    \
        case 6: return fn<2, 0>(__VA_ARGS__); case 7: return fn<2, 1>(__VA_ARGS__); case 8: return fn<2, 2>(__VA_ARGS__);    \
        case 9: return fn<3, 0>(__VA_ARGS__); case 10: return fn<3, 1>(__VA_ARGS__); case 11: return fn<3, 2>(__VA_ARGS__);  \
        case 12: return fn<4, 0>(__VA_ARGS__); case 13: return fn<4, 1>(__VA_ARGS__); case 14: return fn<4, 2>(__VA_ARGS__); \
        case 15: return fn<5, 0>(__VA_ARGS__);   /* lmax = 5: packed rotated body only */                            \
    }                                                                                                        \
    return CELES_EINVAL

int launch_coupling(const celes_ctx* c, cudaStream_t s) { CELES_DISPATCH(launch_coupling_t, c, s); }
int prepare_coupling(celes_ctx* c, int* ctas_per_sm) { CELES_DISPATCH(prepare_coupling_t, c, ctas_per_sm); }

// y = W b (tdiag == nullptr) or out = b - T (W b): pack -> coupling -> finalize, all on stream s.
int run_matvec(celes_ctx* c, const float2* b, float2* out, bool system, cudaStream_t s) {
    const int H = c->nmax / 2;
    const long long nh = (long long)c->N * H;
    const int tb = 256;
    const unsigned gb = (unsigned)((nh + tb - 1) / tb);
    if (c->variant == celes::kRotated) celes::pack_kernel<celes::kRotated><<<gb, tb, 0, s>>>(c->N, H, b, c->bpm);
    else if (c->variant == celes::kDirect) celes::pack_kernel<celes::kDirect><<<gb, tb, 0, s>>>(c->N, H, b, c->bpm);
    else celes::pack_kernel<celes::kRotatedScalar><<<gb, tb, 0, s>>>(c->N, H, b, c->bpm);
    if (cudaGetLastError() != cudaSuccess) return CELES_ECUDA;
    int rc = launch_coupling(c, s);
    if (rc) return rc;
    const float2* td = system ? c->tdiag : nullptr;
    if (c->variant == celes::kRotated) celes::finalize_kernel<celes::kRotated><<<gb, tb, 0, s>>>(c->N, H, c->splits, c->ypart, td, b, out);
    else if (c->variant == celes::kDirect) celes::finalize_kernel<celes::kDirect><<<gb, tb, 0, s>>>(c->N, H, c->splits, c->ypart, td, b, out);
    else celes::finalize_kernel<celes::kRotatedScalar><<<gb, tb, 0, s>>>(c->N, H, c->splits, c->ypart, td, b, out);
    return cudaGetLastError() == cudaSuccess ? CELES_OK : CELES_ECUDA;
}

// Spheres must be disjoint ((A.5) needs |r| < |d|).  Uniform grid of cell edge 2 Rmax: every
// sphere is compared with the spheres of the 27 cells around it.  O(N log N).
bool spheres_disjoint(int N, const double* pos, const double* rad) {
    if (N < 2) return true;
    double rmax = 0.0, lo[3] = {pos[0], pos[1], pos[2]};
    for (int i = 0; i < N; ++i) {
        rmax = std::max(rmax, rad[i]);
        for (int a = 0; a < 3; ++a) lo[a] = std::min(lo[a], pos[3 * i + a]);
    }
    const double cell = std::max(2.0 * rmax, 1e-300);
    struct Key { int64_t c[3]; int i; };
    std::vector<Key> keys(N);
    for (int i = 0; i < N; ++i) {
        for (int a = 0; a < 3; ++a) keys[i].c[a] = (int64_t)std::floor((pos[3 * i + a] - lo[a]) / cell);
        keys[i].i = i;
    }
    auto less = [](const Key& x, const Key& y) {
        if (x.c[0] != y.c[0]) return x.c[0] < y.c[0];
        if (x.c[1] != y.c[1]) return x.c[1] < y.c[1];
        return x.c[2] < y.c[2];
    };
    std::sort(keys.begin(), keys.end(), less);
    for (int a = 0; a < N; ++a) {
        const Key& ka = keys[a];
        for (int64_t dx = -1; dx <= 1; ++dx)
            for (int64_t dy = -1; dy <= 1; ++dy) {
                // the three z-neighbours of (cx+dx, cy+dy) are contiguous in the sorted order
                Key probe{{ka.c[0] + dx, ka.c[1] + dy, ka.c[2] - 1}, 0};
                auto it = std::lower_bound(keys.begin(), keys.end(), probe, less);
                for (; it != keys.end() && it->c[0] == probe.c[0] && it->c[1] == probe.c[1] && it->c[2] <= ka.c[2] + 1; ++it) {
                    const int i = ka.i, j = it->i;
                    if (j <= i) continue;
                    const double ex = pos[3 * i] - pos[3 * j], ey = pos[3 * i + 1] - pos[3 * j + 1],
                                 ez = pos[3 * i + 2] - pos[3 * j + 2];
                    const double rr = rad[i] + rad[j];
                    if (ex * ex + ey * ey + ez * ez < rr * rr) return false;
                }
            }
    }
    return true;
}

void free_precond(celes_ctx* c) {
    cudaFree(c->pc_order); cudaFree(c->pc_grp_offset); cudaFree(c->pc_blk_offset); cudaFree(c->pc_cta_group);
    cudaFree(c->pc_cta_row0); cudaFree(c->pc_blocks); cudaFree(c->pc_tmp);
    c->pc_order = c->pc_grp_offset = c->pc_cta_group = c->pc_cta_row0 = nullptr;
    c->pc_blk_offset = nullptr; c->pc_blocks = c->pc_tmp = nullptr;
    c->pc_ready = false; c->pc_groups = c->pc_max_n = c->pc_ctas = 0; c->pc_elems = 0;
}

void free_ctx(celes_ctx* c) {
    if (!c) return;
    free_precond(c);
    cudaFree(c->kpos); cudaFree(c->tdiag); cudaFree(c->bpm); cudaFree(c->ypart); cudaFree(c->htab); cudaFree(c->host_in); cudaFree(c->host_out);
    cudaFree(c->V); cudaFree(c->rhs); cudaFree(c->tmp); cudaFree(c->partial); cudaFree(c->coef); cudaFree(c->hsum);
    if (c->hhost) cudaFreeHost(c->hhost);
    for (int q = 0; q < 2; ++q) if (c->kry_ev[q]) cudaEventDestroy(c->kry_ev[q]);
    delete c;
}

// z = blockdiag(M_j^{-1}) v  (step 4)
int precond_apply(celes_ctx* c, const float2* v, float2* z, cudaStream_t s) {
    celes::block_gemv_kernel<<<c->pc_ctas, celes::kGemvRows, (size_t)c->pc_max_n * sizeof(float2), s>>>(
        c->nmax, c->pc_cta_group, c->pc_cta_row0, c->pc_grp_offset, c->pc_order, c->pc_blk_offset, c->pc_blocks, v, z);
    return cudaGetLastError() == cudaSuccess ? CELES_OK : CELES_ECUDA;
}

int ensure_krylov(celes_ctx* c, int restart) {
    if (c->V && c->kry_restart >= restart) return CELES_OK;
    cudaFree(c->V); cudaFree(c->rhs); cudaFree(c->tmp); cudaFree(c->partial); cudaFree(c->coef); cudaFree(c->hsum);
    if (c->hhost) cudaFreeHost(c->hhost);
    c->V = nullptr; c->rhs = c->tmp = nullptr; c->partial = c->coef = c->hsum = nullptr; c->hhost = nullptr;
    const size_t n = (size_t)c->N * c->nmax;
    c->dot_blocks = (int)std::min<size_t>((n + celes::kDotBlock - 1) / celes::kDotBlock, (size_t)c->sm_count * 4);
    CU_TRY(cudaMalloc(&c->V, sizeof(float2) * n * (restart + 1)));
    CU_TRY(cudaMalloc(&c->rhs, sizeof(float2) * n));
    CU_TRY(cudaMalloc(&c->tmp, sizeof(float2) * n));
    CU_TRY(cudaMalloc(&c->partial, sizeof(double2) * c->dot_blocks * (restart + 1)));
    CU_TRY(cudaMalloc(&c->coef, sizeof(double2) * (restart + 2)));
    CU_TRY(cudaMalloc(&c->hsum, sizeof(double2) * 2 * (restart + 2)));
    CU_TRY(cudaMallocHost(&c->hhost, sizeof(double2) * 3 * (restart + 2)));
    for (int q = 0; q < 2; ++q)
        if (!c->kry_ev[q]) CU_TRY(cudaEventCreateWithFlags(&c->kry_ev[q], cudaEventDisableTiming));
    c->kry_restart = restart;
    return CELES_OK;
}

// out[0..k) (device) = V[0..k)^H w; optionally accumulated into accum.
int device_dots(celes_ctx* c, long long n, int k, const float2* V, const float2* w, double2* out, double2* accum,
                cudaStream_t s) {
    celes::multi_dot_kernel<<<c->dot_blocks, celes::kDotBlock, 0, s>>>(n, k, V, w, c->partial);
    celes::dots_reduce_kernel<<<k, celes::kReduceThreads, 0, s>>>(c->dot_blocks, k, c->partial, out, accum);
    return cudaGetLastError() == cudaSuccess ? CELES_OK : CELES_ECUDA;
}

int device_axpys(celes_ctx* c, long long n, int k, double alpha, const double2* coef, const float2* V, float2* w,
                 cudaStream_t s) {
    const int blocks = (int)std::min<long long>((n + 255) / 256, (long long)c->sm_count * 8);
    celes::multi_axpy_kernel<<<blocks, 256, sizeof(double2) * k, s>>>(n, k, alpha, coef, V, w);
    return cudaGetLastError() == cudaSuccess ? CELES_OK : CELES_ECUDA;
}

// ||v||_2 on the host (synchronises s)
int device_norm(celes_ctx* c, long long n, const float2* v, double* out, cudaStream_t s) {
    int rc = device_dots(c, n, 1, v, v, c->coef, nullptr, s);
    if (rc) return rc;
    CU_TRY(cudaMemcpyAsync(c->hhost, c->coef, sizeof(double2), cudaMemcpyDeviceToHost, s));
    CU_TRY(cudaStreamSynchronize(s));
    *out = std::sqrt(std::max(0.0, c->hhost[0].x));
    return CELES_OK;
}

// ---- FP32 peak probe kernels -----------------------------------------------------------------------------
template <int VARIANT>
__global__ void __launch_bounds__(256) ffma_probe_kernel(int iters, float seed, float* sink) {
    constexpr int C = 16;                         // independent chains per thread
    float a[C];
#pragma unroll
    for (int c = 0; c < C; ++c) a[c] = seed + (float)(threadIdx.x + c);
    const float m = 0.999f + seed * 1e-9f, d = seed * 1e-3f;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            if (VARIANT == 0) {
#pragma unroll
                for (int c = 0; c < C; ++c) a[c] = fmaf(a[c], m, d);
            } else if (VARIANT == 1) {
#pragma unroll
                for (int c = 0; c < C; ++c) a[c] = fmaf(a[c], 0.99951171875f, d);
            } else {
#pragma unroll
                for (int c = 0; c < C; c += 2) {
                    unsigned long long acc, mm, dd;
                    asm("mov.b64 %0, {%1, %2};" : "=l"(acc) : "f"(a[c]), "f"(a[c + 1]));
                    asm("mov.b64 %0, {%1, %1};" : "=l"(mm) : "f"(m));
                    asm("mov.b64 %0, {%1, %1};" : "=l"(dd) : "f"(d));
                    asm("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(acc) : "l"(mm), "l"(dd));
                    asm("mov.b64 {%0, %1}, %2;" : "=f"(a[c]), "=f"(a[c + 1]) : "l"(acc));
                }
            }
        }
    }
    float t = 0.f;
#pragma unroll
    for (int c = 0; c < C; ++c) t += a[c];
    if (t == 12345.678f) sink[0] = t;             // never true in practice; keeps the chains alive
}

// Variants 3 / 4: packed fma.rn.f32x2 streams shaped like the pair body (a real coefficient times a packed complex
// value added to a packed accumulator, eight independent accumulators), in a fixed instruction order (asm
// volatile).  3: consecutive instructions share no source register (every operand is fetched from the register
// file); 4: eight consecutive instructions share the packed value (operand reuse cache).  They measure what the
// FMA pipe sustains when three register operands per instruction have to be delivered.
template <int SHARE>
__global__ void __launch_bounds__(128) ffma2_operand_probe_kernel(int iters, const float2* __restrict__ in, float* sink) {
    typedef unsigned long long u64;
    u64 R[8], z[4], u[8];
#pragma unroll
    for (int c = 0; c < 8; ++c) {
        const float r = in[(threadIdx.x + c) & 63].x;
        asm("mov.b64 %0, {%1, %1};" : "=l"(R[c]) : "f"(r));
        asm("mov.b64 %0, {%1, %1};" : "=l"(u[c]) : "f"(0.0f));
    }
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        const float2 v = in[(threadIdx.x + 8 + c) & 63];
        asm("mov.b64 %0, {%1, %2};" : "=l"(z[c]) : "f"(v.x), "f"(v.y));
    }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int rep = 0; rep < 4; ++rep)
#pragma unroll
            for (int m = 0; m < 4; ++m)
#pragma unroll
                for (int t = 0; t < 8; ++t) {
                    if (SHARE) asm volatile("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(u[t]) : "l"(R[(t + m) & 7]), "l"(z[m]));
                    else asm volatile("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(u[t]) : "l"(R[(t + m) & 7]), "l"(z[(t + m) & 3]));
                }
    }
    float acc = 0.f;
#pragma unroll
    for (int c = 0; c < 8; ++c) {
        float a, b;
        asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(u[c]));
        acc += a + b;
    }
    if (acc == 12345.678f) sink[0] = acc;
}

}  // namespace

// ---------------------------------------------------------------------------------------------------------
extern "C" {

int celes_nmax(int lmax) {
    if (lmax < CELES_LMAX_MIN || lmax > CELES_LMAX_MAX) return CELES_EINVAL;
    return 2 * lmax * (lmax + 2);
}

const char* celes_strerror(int code) {
    switch (code) {
        case CELES_OK: return "success";
        case CELES_EINVAL: return "invalid argument";
        case CELES_ENOMEM: return "out of memory";
        case CELES_ECUDA: return "CUDA error or no CUDA device";
        case CELES_ENOCONV: return "iterative solver did not converge within max_iters";
    }
    return "unknown error code";
}

int celes_translation_table(int lmax, double* a5_re, double* b5_im) {
    if (lmax < CELES_LMAX_MIN || lmax > CELES_LMAX_MAX || !a5_re || !b5_im) return CELES_EINVAL;
    std::vector<double> a, b;
    if (!celes::build_translation_table(lmax, a, b)) return CELES_EINVAL;
    std::memcpy(a5_re, a.data(), sizeof(double) * a.size());
    std::memcpy(b5_im, b.data(), sizeof(double) * b.size());
    return CELES_OK;
}

int celes_setup(celes_ctx** out, int N, int lmax, const double* pos_xyz, const double* radii, const double* mie_q,
                double k, const celes_options* opt, void* cuda_stream) {
    if (!out) return CELES_EINVAL;
    *out = nullptr;
    if (N < 1 || lmax < CELES_LMAX_MIN || lmax > CELES_LMAX_MAX || !pos_xyz || !radii || !mie_q) return CELES_EINVAL;
    if (!(k > 0.0) || !std::isfinite(k)) return CELES_EINVAL;
    if ((long long)N * celes_nmax(lmax) > (1LL << 31)) return CELES_EINVAL;
    const int nmax = celes_nmax(lmax), H = nmax / 2;
    for (long long t = 0; t < 3LL * N; ++t) if (!std::isfinite(pos_xyz[t])) return CELES_EINVAL;
    for (int i = 0; i < N; ++i) if (!std::isfinite(radii[i]) || !(radii[i] > 0.0)) return CELES_EINVAL;
    for (long long t = 0; t < 4LL * N * lmax; ++t) if (!std::isfinite(mie_q[t])) return CELES_EINVAL;
    const bool skip = opt && opt->skip_overlap_check;
    if (!skip && !spheres_disjoint(N, pos_xyz, radii)) return CELES_EINVAL;
    if (opt && (opt->emitter_tile < 0 || opt->emitter_splits < 0 || opt->emitter_tile > 128)) return CELES_EINVAL;
    if (opt && (opt->translation < 0 || opt->translation > CELES_TRANSLATION_ROTATED_SCALAR)) return CELES_EINVAL;
    if (lmax > 4 && opt && opt->translation != CELES_TRANSLATION_ROTATED) return CELES_EINVAL;   // one body at lmax = 5
    const bool table = opt && opt->hankel == CELES_HANKEL_TABLE;
    if (opt && opt->hankel != CELES_HANKEL_REGISTERS && opt->hankel != CELES_HANKEL_TABLE) return CELES_EINVAL;
    if (table && (opt->translation != CELES_TRANSLATION_ROTATED || !(opt->hankel_dr >= 0.0) || !std::isfinite(opt->hankel_dr)))
        return CELES_EINVAL;

    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { cudaGetLastError(); return CELES_ECUDA; }
    celes_ctx* c = new (std::nothrow) celes_ctx;
    if (!c) return CELES_ENOMEM;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    c->N = N; c->lmax = lmax; c->nmax = nmax; c->k = k;
    int rc = CELES_OK;
    auto fail = [&](int code) { free_ctx(c); return code; };
    if (cudaGetDevice(&c->device) != cudaSuccess) return fail(CELES_ECUDA);
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, c->device) != cudaSuccess) return fail(CELES_ECUDA);
    c->sm_count = prop.multiProcessorCount;
    c->etile = (opt && opt->emitter_tile > 0) ? opt->emitter_tile : 32;
    c->variant = opt ? opt->translation : CELES_TRANSLATION_ROTATED;
    c->rblocks = (N + kBlock - 1) / kBlock;
    if (table) {
        // S2: h_p^(1)(k r) for r from the smallest possible centre distance (two touching spheres of
        // the smallest radius; spheres are disjoint) to the diagonal of the centres' bounding box, spacing dr; FP64
        // on the host, stored FP32 with the derivative (h_p' = h_{p-1} - (p+1)/x h_p, h_0' = -h_1) for Hermite cubics.
        const double dr = opt->hankel_dr > 0.0 ? opt->hankel_dr : 1.0;
        double rmin = radii[0], lo[3] = {pos_xyz[0], pos_xyz[1], pos_xyz[2]}, hi[3] = {pos_xyz[0], pos_xyz[1], pos_xyz[2]};
        for (int i = 0; i < N; ++i) {
            rmin = std::min(rmin, radii[i]);
            for (int a = 0; a < 3; ++a) { lo[a] = std::min(lo[a], pos_xyz[3 * i + a]); hi[a] = std::max(hi[a], pos_xyz[3 * i + a]); }
        }
        const double dmin = 2.0 * rmin;
        const double dmax = std::sqrt((hi[0] - lo[0]) * (hi[0] - lo[0]) + (hi[1] - lo[1]) * (hi[1] - lo[1]) + (hi[2] - lo[2]) * (hi[2] - lo[2]));
        const double nodes_d = std::ceil(std::max(0.0, dmax - dmin) / dr) + 2.0;
        const int P = 2 * lmax + 1;
        if (!(nodes_d * P * sizeof(float4) <= 2.0e9)) return fail(CELES_EINVAL);           // table spacing too fine
        const int nodes = (int)nodes_d;
        std::vector<float4> tab((size_t)nodes * P);
        for (int j = 0; j < nodes; ++j) {
            const double x = k * (dmin + j * dr), dxs = k * dr;
            typedef std::complex<double> cd;
            const cd e = std::exp(cd(0.0, x));
            cd h[16];
            h[0] = cd(0.0, -1.0) * e / x;
            h[1] = -e * cd(x, 1.0) / (x * x);
            for (int p = 1; p + 1 < P; ++p) h[p + 1] = (2.0 * p + 1.0) / x * h[p] - h[p - 1];
            for (int p = 0; p < P; ++p) {
                const cd d = p == 0 ? -h[1] : h[p - 1] - (p + 1.0) / x * h[p];
                tab[(size_t)j * P + p] = make_float4((float)h[p].real(), (float)h[p].imag(), (float)(dxs * d.real()), (float)(dxs * d.imag()));
            }
        }
        if (cudaMalloc(&c->htab, sizeof(float4) * tab.size()) != cudaSuccess) return fail(CELES_ENOMEM);
        if (cudaMemcpy(c->htab, tab.data(), sizeof(float4) * tab.size(), cudaMemcpyHostToDevice) != cudaSuccess) return fail(CELES_ECUDA);
        c->htab_desc.nodes = c->htab;
        c->htab_desc.x0 = (float)(k * dmin);
        c->htab_desc.inv_dx = (float)(1.0 / (k * dr));
        c->htab_desc.last = nodes - 1;
    }
    int ctas_per_sm = 1;
    rc = prepare_coupling(c, &ctas_per_sm);
    if (rc) return fail(rc);
    ctas_per_sm = std::max(1, ctas_per_sm);
    if (opt && opt->emitter_splits > 0) {
        c->splits = std::min(opt->emitter_splits, N);
    } else {
        // Split the emitter sum so that the grid is a whole number of waves (slots = SMs x resident CTAs): among
        // 1..16 waves take the split with the best fill (all CTAs do equal work, so a full last wave means no
        // tail), slightly preferring more waves, with at least 96 emitters per CTA.
        const long long slots = (long long)c->sm_count * ctas_per_sm;
        const long long maxsp = std::max<long long>(1, N / 96);
        long long best = 1;
        double best_score = -1.0;
        for (long long waves = 1; waves <= 16; ++waves) {
            const long long sp = std::min(maxsp, std::max<long long>(1, (waves * slots) / c->rblocks));
            const long long used_waves = (sp * c->rblocks + slots - 1) / slots;
            const double eff = (double)sp * c->rblocks / ((double)used_waves * slots);
            const double score = eff - 0.02 / (double)used_waves;
            if (score > best_score + 1e-12) { best_score = score; best = sp; }
        }
        c->splits = (int)best;
    }
    c->chunk = (N + c->splits - 1) / c->splits;
    c->splits = (N + c->chunk - 1) / c->chunk;

    const size_t n = (size_t)N * nmax;
    c->pos.assign(pos_xyz, pos_xyz + 3 * (size_t)N);
    std::vector<double> kp(3 * (size_t)N);
    for (size_t t = 0; t < kp.size(); ++t) kp[t] = k * pos_xyz[t];
    std::vector<float2> td(n);
    const std::complex<double>* q = reinterpret_cast<const std::complex<double>*>(mie_q);
    for (int i = 0; i < N; ++i)
        for (int tau = 0; tau < 2; ++tau)
            for (int l = 1; l <= lmax; ++l)
                for (int m = -l; m <= l; ++m) {
                    const std::complex<double> v = q[((size_t)i * 2 + tau) * lmax + (l - 1)];
                    td[(size_t)i * nmax + tau * H + (l - 1) * (l + 1) + (m + l)] = make_float2((float)v.real(), (float)v.imag());
                }
#define SETUP_TRY(expr)                                                        \
    do {                                                                       \
        cudaError_t e_ = (expr);                                               \
        if (e_ != cudaSuccess) return fail(e_ == cudaErrorMemoryAllocation ? CELES_ENOMEM : CELES_ECUDA); \
    } while (0)
    SETUP_TRY(cudaMalloc(&c->kpos, sizeof(double) * kp.size()));
    SETUP_TRY(cudaMalloc(&c->tdiag, sizeof(float2) * n));
    SETUP_TRY(cudaMalloc(&c->bpm, sizeof(float2) * n));
    SETUP_TRY(cudaMalloc(&c->ypart, sizeof(float2) * n * c->splits));
    SETUP_TRY(cudaMemcpyAsync(c->kpos, kp.data(), sizeof(double) * kp.size(), cudaMemcpyHostToDevice, s));
    SETUP_TRY(cudaMemcpyAsync(c->tdiag, td.data(), sizeof(float2) * n, cudaMemcpyHostToDevice, s));
    SETUP_TRY(cudaStreamSynchronize(s));
#undef SETUP_TRY
    *out = c;
    return CELES_OK;
}

int celes_coupling_matvec(celes_ctx* ctx, const void* b_dev, void* y_dev, void* cuda_stream) {
    if (!ctx || !b_dev || !y_dev || b_dev == y_dev) return CELES_EINVAL;
    return run_matvec(ctx, (const float2*)b_dev, (float2*)y_dev, false, (cudaStream_t)cuda_stream);
}

int celes_system_matvec(celes_ctx* ctx, const void* b_dev, void* out_dev, void* cuda_stream) {
    if (!ctx || !b_dev || !out_dev || b_dev == out_dev) return CELES_EINVAL;
    return run_matvec(ctx, (const float2*)b_dev, (float2*)out_dev, true, (cudaStream_t)cuda_stream);
}

static int matvec_host(celes_ctx* ctx, const void* b_host, void* y_host, bool system, void* cuda_stream) {
    if (!ctx || !b_host || !y_host) return CELES_EINVAL;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const size_t bytes = sizeof(float2) * (size_t)ctx->N * ctx->nmax;
    if (!ctx->host_in) {                       // device staging buffers of the host entry points, kept with the context
        CU_TRY(cudaMalloc(&ctx->host_in, bytes));
        if (cudaMalloc(&ctx->host_out, bytes) != cudaSuccess) { cudaFree(ctx->host_in); ctx->host_in = nullptr; return CELES_ENOMEM; }
    }
    int rc = CELES_OK;
    if (cudaMemcpyAsync(ctx->host_in, b_host, bytes, cudaMemcpyHostToDevice, s) != cudaSuccess) rc = CELES_ECUDA;
    if (!rc) rc = run_matvec(ctx, ctx->host_in, ctx->host_out, system, s);
    if (!rc && cudaMemcpyAsync(y_host, ctx->host_out, bytes, cudaMemcpyDeviceToHost, s) != cudaSuccess) rc = CELES_ECUDA;
    if (cudaStreamSynchronize(s) != cudaSuccess && !rc) rc = CELES_ECUDA;
    return rc;
}

int celes_coupling_matvec_host(celes_ctx* ctx, const void* b_host, void* y_host, void* cuda_stream) {
    return matvec_host(ctx, b_host, y_host, false, cuda_stream);
}

int celes_system_matvec_host(celes_ctx* ctx, const void* b_host, void* out_host, void* cuda_stream) {
    return matvec_host(ctx, b_host, out_host, true, cuda_stream);
}

int celes_launch_config(const celes_ctx* ctx, int* receiver_blocks, int* emitter_splits, int* block_threads,
                        int* emitter_tile) {
    if (!ctx) return CELES_EINVAL;
    if (receiver_blocks) *receiver_blocks = ctx->rblocks;
    if (emitter_splits) *emitter_splits = ctx->splits;
    if (block_threads) *block_threads = kBlock;
    if (emitter_tile) *emitter_tile = ctx->etile;
    return CELES_OK;
}

}  // extern "C"

namespace {
// BiCGSTAB (van der Vorst; the paper's second solver) on M x = T a_in, optionally right-preconditioned
// with the block-diagonal operator.  Three small device->host copies per iteration (the inner products that define
// alpha, omega and rho); every vector operation is a device kernel.  The recursive residual only proposes
// convergence: the TRUE residual rhs - M x is recomputed then and decides (as in the GMRES path, reading R14);
// if it disagrees, or on a breakdown (rho = 0, <r^,v> = 0, <t,t> = 0), the iteration restarts from the true residual.
int solve_bicgstab(celes_ctx* ctx, float2* x, bool pc, double rtol, int max_iters, double fnorm, cudaStream_t s,
                   int& iterations, int& matvecs, int& converged, double& rel, const std::function<void(double)>& push_hist) {
    typedef std::complex<double> cd;
    const long long n = (long long)ctx->N * ctx->nmax;
    const int eb = (int)std::min<long long>((n + 255) / 256, (long long)ctx->sm_count * 8);
    float2* V = ctx->V;
    float2 *rhat = V, *r = V + n, *p = V + 2 * n, *v = V + 3 * n, *sv = V + 4 * n, *t = V + 5 * n, *phat = V + 6 * n,
           *shat = V + 7 * n;
    auto d2 = [](cd z) { return make_double2(z.real(), z.imag()); };
    auto fetch = [&](int k, cd* out) -> int {          // hsum[0..k) -> host
        CU_TRY(cudaMemcpyAsync(ctx->hhost, ctx->hsum, sizeof(double2) * k, cudaMemcpyDeviceToHost, s));
        CU_TRY(cudaStreamSynchronize(s));
        for (int q = 0; q < k; ++q) out[q] = cd(ctx->hhost[q].x, ctx->hhost[q].y);
        return CELES_OK;
    };
    int rc = CELES_OK, restarts = 0;
    while (true) {
        rc = run_matvec(ctx, x, ctx->tmp, true, s);                         // true residual
        if (rc) return rc;
        ++matvecs;
        celes::sub_kernel<<<eb, 256, 0, s>>>(n, ctx->rhs, ctx->tmp, r);
        double beta0 = 0.0;
        rc = device_norm(ctx, n, r, &beta0, s);
        if (rc) return rc;
        rel = beta0 / fnorm;
        push_hist(rel);
        if (rel <= rtol) { converged = 1; return CELES_OK; }
        if (iterations >= max_iters || ++restarts > 50) return CELES_ENOCONV;
        if (!std::isfinite(rel)) return CELES_ECUDA;
        CU_TRY(cudaMemcpyAsync(rhat, r, sizeof(float2) * n, cudaMemcpyDeviceToDevice, s));
        CU_TRY(cudaMemsetAsync(p, 0, sizeof(float2) * n, s));
        CU_TRY(cudaMemsetAsync(v, 0, sizeof(float2) * n, s));
        cd rho = 1.0, alpha = 1.0, omega = 1.0, rho_new = cd(beta0 * beta0, 0.0);
        bool first = true;
        while (iterations < max_iters) {
            const cd beta = first ? cd(0.0) : (rho_new / rho) * (alpha / omega);
            // p = r + beta (p - omega v)
            celes::lincomb_kernel<<<eb, 256, 0, s>>>(n, d2(1.0), r, d2(beta), p, d2(-beta * omega), v, p);
            first = false;
            const float2* pin = p;
            if (pc) { rc = precond_apply(ctx, p, phat, s); if (rc) return rc; pin = phat; }
            rc = run_matvec(ctx, pin, v, true, s);
            if (rc) return rc;
            ++matvecs;
            rc = device_dots(ctx, n, 1, rhat, v, ctx->hsum, nullptr, s);     // <r^, v>
            if (rc) return rc;
            cd dv[2];
            rc = fetch(1, dv);
            if (rc) return rc;
            if (dv[0] == cd(0.0)) break;                                     // breakdown: restart
            alpha = rho_new / dv[0];
            celes::lincomb_kernel<<<eb, 256, 0, s>>>(n, d2(1.0), r, d2(-alpha), v, d2(0.0), nullptr, sv);   // s = r - alpha v
            const float2* sin_ = sv;
            if (pc) { rc = precond_apply(ctx, sv, shat, s); if (rc) return rc; sin_ = shat; }
            rc = run_matvec(ctx, sin_, t, true, s);
            if (rc) return rc;
            ++matvecs; ++iterations;
            rc = device_dots(ctx, n, 2, sv, t, ctx->hsum, nullptr, s);       // <s, t>, <t, t>   (sv and t are adjacent)
            if (rc) return rc;
            rc = fetch(2, dv);
            if (rc) return rc;
            if (dv[1].real() <= 0.0) {                                      // t = 0: s is the residual, x += alpha p^
                celes::lincomb_kernel<<<eb, 256, 0, s>>>(n, d2(1.0), x, d2(alpha), pin, d2(0.0), nullptr, x);
                break;
            }
            omega = std::conj(dv[0]) / dv[1].real();                         // <t, s> / <t, t>
            celes::lincomb_kernel<<<eb, 256, 0, s>>>(n, d2(1.0), x, d2(alpha), pin, d2(omega), sin_, x);
            celes::lincomb_kernel<<<eb, 256, 0, s>>>(n, d2(1.0), sv, d2(-omega), t, d2(0.0), nullptr, r);   // r = s - omega t
            rho = rho_new;
            rc = device_dots(ctx, n, 2, rhat, r, ctx->hsum, nullptr, s);     // <r^, r>, <r, r>   (rhat and r are adjacent)
            if (rc) return rc;
            rc = fetch(2, dv);
            if (rc) return rc;
            rho_new = dv[0];
            const double est = std::sqrt(std::max(0.0, dv[1].real())) / fnorm;
            push_hist(est);
            if (est <= rtol || rho_new == cd(0.0) || omega == cd(0.0) || !std::isfinite(est)) break;
        }
    }
}

}  // namespace

extern "C" {

// Restarted GMRES (Saad & Schultz, the paper's ref. [26]) on M x = T a_in, unpreconditioned,
// classical Gram-Schmidt with one re-orthogonalisation pass (CGS2): the j+1 inner products of a pass are ONE
// kernel, their coefficients stay on the device for the update, and one small device->host copy per inner
// iteration brings the Hessenberg column to the host, where Givens rotations track the residual estimate; the
// device work of the next column is enqueued before the host waits for that copy (one column of look-ahead).
// The TRUE residual is recomputed at every restart and decides convergence (reading R14).
int celes_solve(celes_ctx* ctx, const void* a_in_dev, void* x_dev, const celes_solve_opts* o, celes_solve_info* info,
                void* cuda_stream) {
    if (!ctx || !a_in_dev || !x_dev) return CELES_EINVAL;
    const int method = o ? o->method : CELES_GMRES;
    const int restart = (o && o->restart > 0) ? o->restart : 30;
    const double rtol = (o && o->rtol > 0.0) ? o->rtol : 1e-4;
    const int max_iters = (o && o->max_iters > 0) ? o->max_iters : 1000;
    const bool pc = o && o->precond == CELES_PRECOND_BLOCKDIAG;
    if ((method != CELES_GMRES && method != CELES_BICGSTAB) || restart > 1024) return CELES_EINVAL;
    if (o && o->precond != CELES_PRECOND_NONE && o->precond != CELES_PRECOND_BLOCKDIAG) return CELES_EINVAL;
    if (pc && !ctx->pc_ready) return CELES_EINVAL;            // celes_precond_setup first
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const auto t_start = std::chrono::steady_clock::now();
    int rc = ensure_krylov(ctx, method == CELES_BICGSTAB ? std::max(restart, 8) : restart);
    if (rc) return rc;
    const long long n = (long long)ctx->N * ctx->nmax;
    const int eb = (int)std::min<long long>((n + 255) / 256, (long long)ctx->sm_count * 8);
    float2* x = (float2*)x_dev;
    float2* V = ctx->V;
    typedef std::complex<double> cd;

    int iterations = 0, matvecs = 0, n_hist = 0, converged = 0;
    double rel = 0.0;
    if (info) std::memset(info, 0, sizeof(*info));
    auto push_hist = [&](double v) { if (info && n_hist < CELES_MAX_HISTORY) info->history[n_hist++] = v; };
    auto finish = [&](int code) {
        if (info) {
            info->iterations = iterations; info->matvecs = matvecs; info->converged = converged;
            info->rel_residual = rel; info->n_history = n_hist;
            info->seconds = std::chrono::duration<double>(std::chrono::steady_clock::now() - t_start).count();
        }
        return code;
    };

    // rhs = T a_in (eq. 8)
    celes::tapply_kernel<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(n, ctx->tdiag, (const float2*)a_in_dev, ctx->rhs);
    double fnorm = 0.0;
    rc = device_norm(ctx, n, ctx->rhs, &fnorm, s);
    if (rc) return finish(rc);
    if (fnorm == 0.0) {                       // zero right-hand side: x = 0
        CU_TRY(cudaMemsetAsync(x, 0, sizeof(float2) * n, s));
        CU_TRY(cudaStreamSynchronize(s));
        converged = 1;
        return finish(CELES_OK);
    }

    if (method == CELES_BICGSTAB)
        return finish(solve_bicgstab(ctx, x, pc, rtol, max_iters, fnorm, s, iterations, matvecs, converged, rel, push_hist));

    std::vector<cd> Hm((size_t)(restart + 1) * restart), g(restart + 1), cs(restart), sn(restart), yv(restart);
    while (true) {
        // true residual r = rhs - M x  -> V_0
        rc = run_matvec(ctx, x, ctx->tmp, true, s);
        if (rc) return finish(rc);
        ++matvecs;
        celes::sub_kernel<<<eb, 256, 0, s>>>(n, ctx->rhs, ctx->tmp, V);
        double beta = 0.0;
        rc = device_norm(ctx, n, V, &beta, s);
        if (rc) return finish(rc);
        rel = beta / fnorm;
        if (n_hist == 0) push_hist(rel);
        if (rel <= rtol) { converged = 1; return finish(CELES_OK); }
        if (iterations >= max_iters) return finish(CELES_ENOCONV);
        if (!std::isfinite(rel)) return finish(CELES_ECUDA);
        // V_0 = r / beta  (coef[0] still holds <r,r>)
        celes::scale_by_inv_norm_kernel<<<eb, 256, 0, s>>>(n, ctx->coef, V, V);
        std::fill(g.begin(), g.end(), cd(0.0));
        g[0] = beta;
        // Arnoldi with one column of look-ahead: the device work of column j+1 (it only needs v_{j+1}, which is
        // normalised on the device) is enqueued BEFORE the host waits for the Hessenberg column j, so the Givens
        // update and the copy latency overlap the next matvec.  Convergence is seen one column late at worst:
        // the column already enqueued is then simply not used.
        const int hs = ctx->kry_restart + 2;                   // stride of the two hsum / hhost halves (as allocated)
        auto enqueue_column = [&](int jc) -> int {
            float2* w = V + (size_t)(jc + 1) * n;
            double2* hsum = ctx->hsum + (size_t)(jc & 1) * hs;
            int r2;
            if (pc) {                                          // right preconditioning: w = M (P^{-1} v_j)
                r2 = precond_apply(ctx, V + (size_t)jc * n, ctx->pc_tmp, s);
                if (r2) return r2;
                r2 = run_matvec(ctx, ctx->pc_tmp, w, true, s);
            } else {
                r2 = run_matvec(ctx, V + (size_t)jc * n, w, true, s);
            }
            if (r2) return r2;
            ++matvecs;
            CU_TRY(cudaMemsetAsync(hsum, 0, sizeof(double2) * (jc + 2), s));
            for (int pass = 0; pass < 2; ++pass) {
                r2 = device_dots(ctx, n, jc + 1, V, w, ctx->coef, hsum, s);
                if (r2) return r2;
                r2 = device_axpys(ctx, n, jc + 1, -1.0, ctx->coef, V, w, s);
                if (r2) return r2;
            }
            r2 = device_dots(ctx, n, 1, w, w, hsum + (jc + 1), nullptr, s);
            if (r2) return r2;
            celes::scale_by_inv_norm_kernel<<<eb, 256, 0, s>>>(n, hsum + (jc + 1), w, w);
            CU_TRY(cudaMemcpyAsync(ctx->hhost + (size_t)(jc & 1) * hs, hsum, sizeof(double2) * (jc + 2), cudaMemcpyDeviceToHost, s));
            CU_TRY(cudaEventRecord(ctx->kry_ev[jc & 1], s));
            return CELES_OK;
        };
        int j = 0, enq = 0;
        if (iterations < max_iters) {
            rc = enqueue_column(0);
            if (rc) return finish(rc);
            enq = 1;
        }
        while (j < enq) {
            if (enq < restart && iterations + (enq - j) < max_iters) {      // look-ahead
                rc = enqueue_column(enq);
                if (rc) return finish(rc);
                ++enq;
            }
            CU_TRY(cudaEventSynchronize(ctx->kry_ev[j & 1]));
            ++iterations;
            const double2* hh = ctx->hhost + (size_t)(j & 1) * hs;
            // Hessenberg column j, Givens rotations
            cd* col = &Hm[(size_t)j * (restart + 1)];
            for (int i = 0; i <= j; ++i) col[i] = cd(hh[i].x, hh[i].y);
            const double hnext = std::sqrt(std::max(0.0, hh[j + 1].x));
            for (int i = 0; i < j; ++i) {
                const cd t = cs[i] * col[i] + sn[i] * col[i + 1];
                col[i + 1] = -std::conj(sn[i]) * col[i] + cs[i] * col[i + 1];
                col[i] = t;
            }
            const double denom = std::sqrt(std::norm(col[j]) + hnext * hnext);
            if (denom == 0.0) break;                               // exact breakdown: drop the column
            cs[j] = std::abs(col[j]) / denom;                       // real c, complex s (|c|^2 + |s|^2 = 1)
            const cd phase = (std::abs(col[j]) > 0.0) ? col[j] / std::abs(col[j]) : cd(1.0);
            sn[j] = phase * hnext / denom;
            col[j] = phase * denom;
            g[j + 1] = -std::conj(sn[j]) * g[j];
            g[j] = cs[j] * g[j];
            const double est = std::abs(g[j + 1]) / fnorm;
            push_hist(est);
            ++j;
            if (est <= rtol || hnext == 0.0) break;
        }
        double2* hup = ctx->hhost + 2 * (size_t)hs;            // third part of the pinned buffer: coefficient upload
        // back substitution R y = g, x += V y
        for (int i = j - 1; i >= 0; --i) {
            cd acc = g[i];
            for (int q = i + 1; q < j; ++q) acc -= Hm[(size_t)q * (restart + 1) + i] * yv[q];
            yv[i] = acc / Hm[(size_t)i * (restart + 1) + i];
        }
        for (int i = 0; i < j; ++i) hup[i] = make_double2(yv[i].real(), yv[i].imag());
        CU_TRY(cudaMemcpyAsync(ctx->coef, hup, sizeof(double2) * j, cudaMemcpyHostToDevice, s));
        if (j > 0 && pc) {                                     // x += P^{-1} (V y)
            CU_TRY(cudaMemsetAsync(ctx->tmp, 0, sizeof(float2) * n, s));
            rc = device_axpys(ctx, n, j, 1.0, ctx->coef, V, ctx->tmp, s);
            if (rc) return finish(rc);
            rc = precond_apply(ctx, ctx->tmp, ctx->pc_tmp, s);
            if (rc) return finish(rc);
            celes::add_kernel<<<eb, 256, 0, s>>>(n, ctx->pc_tmp, x);
        } else if (j > 0) {
            rc = device_axpys(ctx, n, j, 1.0, ctx->coef, V, x, s);
            if (rc) return finish(rc);
        }
        CU_TRY(cudaStreamSynchronize(s));      // hhost is reused by the next cycle
    }
}

int celes_partition(int N, const double* pos_xyz, const double* edge_xyz, int* group_of, int* n_groups) {
    if (N < 1 || !pos_xyz || !edge_xyz || !group_of) return CELES_EINVAL;
    celes::Partition part;
    if (!celes::build_partition(N, pos_xyz, edge_xyz, part)) return CELES_EINVAL;
    std::memcpy(group_of, part.group_of.data(), sizeof(int) * (size_t)N);
    if (n_groups) *n_groups = part.n_groups();
    return CELES_OK;
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

int celes_far_field(celes_ctx* ctx, const void* b_dev, int n_dir, const double* alpha, const double* beta, void* g_dev,
                    void* cuda_stream) {
    if (!ctx || !b_dev || !g_dev || n_dir < 1 || !alpha || !beta || n_dir > (1 << 29)) return CELES_EINVAL;
    for (int d = 0; d < n_dir; ++d)
        if (!std::isfinite(alpha[d]) || !std::isfinite(beta[d])) return CELES_EINVAL;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const int nmax = ctx->nmax, rows = 2 * n_dir, gx = (rows + celes::kFarThreads - 1) / celes::kFarThreads;
    // split the sphere sum so that the grid has about four CTAs per SM-slot pair, at least 4 tiles per CTA
    int splits = std::max(1, std::min((8 * ctx->sm_count + gx - 1) / gx, std::max(1, ctx->N / (4 * celes::kFarTile))));
    const int chunk = ((ctx->N + splits - 1) / splits + celes::kFarTile - 1) / celes::kFarTile * celes::kFarTile;
    splits = (ctx->N + chunk - 1) / chunk;
    double *d_ang = nullptr, *d_dir = nullptr;
    float2 *d_coef = nullptr, *d_part = nullptr;
    int rc = CELES_OK;
    if (cudaMalloc(&d_ang, sizeof(double) * 2 * (size_t)n_dir) != cudaSuccess ||
        cudaMalloc(&d_dir, sizeof(double) * 3 * (size_t)n_dir) != cudaSuccess ||
        cudaMalloc(&d_coef, sizeof(float2) * (size_t)rows * nmax) != cudaSuccess ||
        cudaMalloc(&d_part, sizeof(float2) * (size_t)rows * splits) != cudaSuccess) rc = CELES_ENOMEM;
    if (!rc && (cudaMemcpyAsync(d_ang, alpha, sizeof(double) * n_dir, cudaMemcpyHostToDevice, s) != cudaSuccess ||
                cudaMemcpyAsync(d_ang + n_dir, beta, sizeof(double) * n_dir, cudaMemcpyHostToDevice, s) != cudaSuccess)) rc = CELES_ECUDA;
    if (!rc) {
        celes::far_field_coefficients_kernel<<<(n_dir + 127) / 128, 128, 0, s>>>(ctx->lmax, n_dir, d_ang, d_ang + n_dir, d_coef, d_dir);
        const float2* b = (const float2*)b_dev;
        dim3 grid(gx, splits);
        switch (ctx->lmax) {
            case 1: celes::far_field_kernel<6><<<grid, celes::kFarThreads, 0, s>>>(ctx->N, chunk, rows, ctx->kpos, b, d_coef, d_dir, d_part); break;
            case 2: celes::far_field_kernel<16><<<grid, celes::kFarThreads, 0, s>>>(ctx->N, chunk, rows, ctx->kpos, b, d_coef, d_dir, d_part); break;
            case 3: celes::far_field_kernel<30><<<grid, celes::kFarThreads, 0, s>>>(ctx->N, chunk, rows, ctx->kpos, b, d_coef, d_dir, d_part); break;
            case 4: celes::far_field_kernel<48><<<grid, celes::kFarThreads, 0, s>>>(ctx->N, chunk, rows, ctx->kpos, b, d_coef, d_dir, d_part); break;
            case 5: celes::far_field_kernel<70><<<grid, celes::kFarThreads, 0, s>>>(ctx->N, chunk, rows, ctx->kpos, b, d_coef, d_dir, d_part); break;
            default: rc = CELES_EINVAL;
        }
        if (!rc) celes::far_field_reduce_kernel<<<(rows + 255) / 256, 256, 0, s>>>(rows, splits, d_part, (float2*)g_dev);
        if (!rc && cudaGetLastError() != cudaSuccess) rc = CELES_ECUDA;
    }
    if (cudaStreamSynchronize(s) != cudaSuccess && !rc) rc = CELES_ECUDA;
    cudaFree(d_ang); cudaFree(d_dir); cudaFree(d_coef); cudaFree(d_part);
    return rc;
}

int celes_gaussian_beam(celes_ctx* ctx, const celes_beam* beam, void* a_in_dev, void* cuda_stream) {
    if (!ctx || !beam || !a_in_dev) return CELES_EINVAL;
    const int n_beta = beam->n_beta > 0 ? beam->n_beta : 400;
    if (!(beam->waist > 0.0) || !std::isfinite(beam->waist) || n_beta > 100000) return CELES_EINVAL;
    for (int a = 0; a < 3; ++a) if (!std::isfinite(beam->center[a])) return CELES_EINVAL;
    if (!std::isfinite(beam->alpha_G) || !std::isfinite(beam->E0_re) || !std::isfinite(beam->E0_im)) return CELES_EINVAL;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    std::vector<double> sb, cb;
    std::vector<double2> cminus, cplus;
    celes::gaussian_beam_tables(ctx->lmax, n_beta, ctx->k, beam->waist, sb, cb, cminus, cplus);
    double *d_sb = nullptr, *d_cb = nullptr;
    double2 *d_cm = nullptr, *d_cp = nullptr;
    int rc = CELES_OK;
    if (cudaMalloc(&d_sb, sizeof(double) * n_beta) != cudaSuccess || cudaMalloc(&d_cb, sizeof(double) * n_beta) != cudaSuccess ||
        cudaMalloc(&d_cm, sizeof(double2) * cminus.size()) != cudaSuccess ||
        cudaMalloc(&d_cp, sizeof(double2) * cplus.size()) != cudaSuccess) rc = CELES_ENOMEM;
    if (!rc && (cudaMemcpyAsync(d_sb, sb.data(), sizeof(double) * n_beta, cudaMemcpyHostToDevice, s) != cudaSuccess ||
                cudaMemcpyAsync(d_cb, cb.data(), sizeof(double) * n_beta, cudaMemcpyHostToDevice, s) != cudaSuccess ||
                cudaMemcpyAsync(d_cm, cminus.data(), sizeof(double2) * cminus.size(), cudaMemcpyHostToDevice, s) != cudaSuccess ||
                cudaMemcpyAsync(d_cp, cplus.data(), sizeof(double2) * cplus.size(), cudaMemcpyHostToDevice, s) != cudaSuccess)) rc = CELES_ECUDA;
    if (!rc) {
        const long long total = (long long)ctx->N * ctx->nmax;
        celes::gaussian_beam_kernel<<<(unsigned)((total + 127) / 128), 128, 0, s>>>(
            ctx->N, ctx->lmax, n_beta, ctx->kpos, ctx->k * beam->center[0], ctx->k * beam->center[1], ctx->k * beam->center[2],
            beam->alpha_G, make_double2(beam->E0_re, beam->E0_im), d_sb, d_cb, d_cm, d_cp, (float2*)a_in_dev);
        if (cudaGetLastError() != cudaSuccess) rc = CELES_ECUDA;
    }
    if (cudaStreamSynchronize(s) != cudaSuccess && !rc) rc = CELES_ECUDA;
    cudaFree(d_sb); cudaFree(d_cb); cudaFree(d_cm); cudaFree(d_cp);
    return rc;
}

int celes_scattered_field(celes_ctx* ctx, const void* b_dev, int n_pts, const double* pts_xyz, void* e_dev, void* cuda_stream) {
    if (!ctx || !b_dev || !e_dev || !pts_xyz || n_pts < 1) return CELES_EINVAL;
    for (long long t = 0; t < 3LL * n_pts; ++t) if (!std::isfinite(pts_xyz[t])) return CELES_EINVAL;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    std::vector<double> kp(3 * (size_t)n_pts);
    for (size_t t = 0; t < kp.size(); ++t) kp[t] = ctx->k * pts_xyz[t];
    double* d_pts = nullptr;
    CU_TRY(cudaMalloc(&d_pts, sizeof(double) * kp.size()));
    int rc = CELES_OK;
    if (cudaMemcpyAsync(d_pts, kp.data(), sizeof(double) * kp.size(), cudaMemcpyHostToDevice, s) != cudaSuccess) rc = CELES_ECUDA;
    if (!rc) {
        const int grid = (n_pts + celes::kNearThreads - 1) / celes::kNearThreads;
        const float2* b = (const float2*)b_dev;
        float2* E = (float2*)e_dev;
        switch (ctx->lmax) {
            case 1: celes::near_field_kernel<1><<<grid, celes::kNearThreads, 0, s>>>(ctx->N, n_pts, ctx->kpos, b, d_pts, E); break;
            case 2: celes::near_field_kernel<2><<<grid, celes::kNearThreads, 0, s>>>(ctx->N, n_pts, ctx->kpos, b, d_pts, E); break;
            case 3: celes::near_field_kernel<3><<<grid, celes::kNearThreads, 0, s>>>(ctx->N, n_pts, ctx->kpos, b, d_pts, E); break;
            case 4: celes::near_field_kernel<4><<<grid, celes::kNearThreads, 0, s>>>(ctx->N, n_pts, ctx->kpos, b, d_pts, E); break;
            case 5: celes::near_field_kernel<5><<<grid, celes::kNearThreads, 0, s>>>(ctx->N, n_pts, ctx->kpos, b, d_pts, E); break;
            default: rc = CELES_EINVAL;
        }
        if (!rc && cudaGetLastError() != cudaSuccess) rc = CELES_ECUDA;
    }
    if (cudaStreamSynchronize(s) != cudaSuccess && !rc) rc = CELES_ECUDA;
    cudaFree(d_pts);
    return rc;
}

void celes_destroy(celes_ctx* ctx) { free_ctx(ctx); }

int celes_fp32_peak_probe(int variant, int iters, double* flops_per_s, double* milliseconds, void* cuda_stream) {
    if (variant < 0 || variant > 4 || iters < 1) return CELES_EINVAL;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { cudaGetLastError(); return CELES_ECUDA; }
    cudaStream_t s = (cudaStream_t)cuda_stream;
    int dev = 0;
    cudaDeviceProp prop;
    CU_TRY(cudaGetDevice(&dev));
    CU_TRY(cudaGetDeviceProperties(&prop, dev));
    float* sink = nullptr;
    CU_TRY(cudaMalloc(&sink, sizeof(float)));
    float2* zeros = nullptr;
    if (cudaMalloc(&zeros, 64 * sizeof(float2)) != cudaSuccess) { cudaFree(sink); return CELES_ENOMEM; }
    cudaMemsetAsync(zeros, 0, 64 * sizeof(float2), s);
    const bool operand = variant >= 3;
    const int blocks = prop.multiProcessorCount * (operand ? 4 : 8), threads = operand ? 128 : 256;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    auto launch = [&](int it) {
        if (variant == 0) ffma_probe_kernel<0><<<blocks, threads, 0, s>>>(it, 1.0f, sink);
        else if (variant == 1) ffma_probe_kernel<1><<<blocks, threads, 0, s>>>(it, 1.0f, sink);
        else if (variant == 2) ffma_probe_kernel<2><<<blocks, threads, 0, s>>>(it, 1.0f, sink);
        else if (variant == 3) ffma2_operand_probe_kernel<0><<<blocks, threads, 0, s>>>(it, zeros, sink);
        else ffma2_operand_probe_kernel<1><<<blocks, threads, 0, s>>>(it, zeros, sink);
    };
    launch(std::max(1, iters / 10));              // warm-up
    cudaEventRecord(e0, s);
    launch(iters);
    cudaEventRecord(e1, s);
    int rc = CELES_OK;
    if (cudaEventSynchronize(e1) != cudaSuccess || cudaGetLastError() != cudaSuccess) rc = CELES_ECUDA;
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(sink);
    cudaFree(zeros);
    const double fmas = (double)blocks * threads * (operand ? 256.0 : 128.0) * (double)iters;   // FMAs per thread and iteration
    if (flops_per_s) *flops_per_s = 2.0 * fmas / (ms * 1e-3);
    if (milliseconds) *milliseconds = ms;
    return rc;
}

}  // extern "C"
