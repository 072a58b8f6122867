// fields.cu -- the steps either side of the solve: celes_gaussian_beam (Appendix C), celes_far_field (A.12, D.1-D.3)
// and celes_scattered_field (eq. 3 with (A.2)).  Kernels in gaussian_beam.cuh, far_field.cuh, near_field.cuh.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <mutex>
#include <vector>

#include "ctx.h"
#include "packed_math.cuh"
#include "far_field.cuh"
#include "gaussian_beam.cuh"
#include "near_field.cuh"

namespace {

// Device scratch of the field calls, kept with the context: grows when a call needs more (the only time these calls
// synchronise the stream and touch the allocator), is reused otherwise.  Pieces are carved at 256-byte boundaries.
struct Scratch {
    celes_ctx* ctx;
    size_t used = 0;
    explicit Scratch(celes_ctx* c) : ctx(c) {}
    static size_t align(size_t b) { return (b + 255) & ~(size_t)255; }
    int reserve(size_t total, cudaStream_t s) {
        if (total <= ctx->scratch_bytes) return CELES_OK;
        if (cudaStreamSynchronize(s) != cudaSuccess) return CELES_ECUDA;      // earlier calls may still read the old block
        cudaFree(ctx->scratch);
        ctx->scratch = nullptr; ctx->scratch_bytes = 0;
        if (cudaMalloc(&ctx->scratch, total) != cudaSuccess) { cudaGetLastError(); return CELES_ENOMEM; }
        ctx->scratch_bytes = total;
        return CELES_OK;
    }
    template <class T> T* take(size_t count) {
        T* p = reinterpret_cast<T*>(static_cast<char*>(ctx->scratch) + used);
        used += align(sizeof(T) * count);
        return p;
    }
};

// ---- static scratch of celes_far_field_noalloc -----------------------------------------------------------------------
// One file-scope device array, held by every GPU that loads the library until the process exits (5 MiB), cut into fixed
// pieces sized for CELES_FAR_FIELD_NOALLOC_MAX_DIR directions and the largest nmax (70, lmax = 5).  In HOST code the
// name g_far_static is only a stand-in for the symbol, not a device address: the address comes from
// cudaGetSymbolAddress, looked up once per device in far_static_scratch_address() below (called by celes_setup with the
// context's device current) and kept in the context.
constexpr size_t kFarStaticBytes = 5u << 20;
constexpr size_t kFarStaticAngOff = 0;                                                               // [2][max_dir] double
constexpr size_t kFarStaticDirOff = kFarStaticAngOff + sizeof(double) * 2 * CELES_FAR_FIELD_NOALLOC_MAX_DIR;    // [max_dir][3] double
constexpr size_t kFarStaticCoefOff = kFarStaticDirOff + sizeof(double) * 3 * CELES_FAR_FIELD_NOALLOC_MAX_DIR;   // [2 max_dir][70] float2
constexpr size_t kFarStaticPartOff = kFarStaticCoefOff + sizeof(float2) * 2 * CELES_FAR_FIELD_NOALLOC_MAX_DIR * 70;
constexpr size_t kFarStaticPartCapacity = (kFarStaticBytes - kFarStaticPartOff) / sizeof(float2);    // split partial sums
static_assert(kFarStaticDirOff % 256 == 0 && kFarStaticCoefOff % 256 == 0 && kFarStaticPartOff % 256 == 0, "pieces stay 256-byte aligned");
static_assert(kFarStaticPartOff < kFarStaticBytes, "the array holds the tables");
static __device__ __align__(256) unsigned char g_far_static[kFarStaticBytes];

constexpr int kMaxDevices = 64;
std::mutex g_far_static_mutex;
void* g_far_static_addr[kMaxDevices] = {};     // device address of g_far_static on device d (null: not looked up yet)

}  // namespace

// Device address of the static scratch on the CURRENT device (which must be `device`); one cudaGetSymbolAddress per device
// and process.  Allocates nothing: the array is part of the library's device image.
int celes::host::far_static_scratch_address(int device, void** out) {
    if (!out || device < 0 || device >= kMaxDevices) return CELES_EINVAL;
    std::lock_guard<std::mutex> lock(g_far_static_mutex);
    if (g_far_static_addr[device] == nullptr) {
        void* p = nullptr;
        if (cudaGetSymbolAddress(&p, g_far_static) != cudaSuccess || p == nullptr) { cudaGetLastError(); return CELES_ECUDA; }
        g_far_static_addr[device] = p;
    }
    *out = g_far_static_addr[device];
    return CELES_OK;
}

extern "C" {

int celes_far_field(celes_ctx* ctx, const void* b_dev, int n_dir, const double* alpha, const double* beta, void* g_dev,
                    void* cuda_stream) {
    if (!ctx || !b_dev || !g_dev || n_dir < 1 || !alpha || !beta || n_dir > (1 << 29)) return CELES_EINVAL;
    for (int d = 0; d < n_dir; ++d)
        if (!std::isfinite(alpha[d]) || !std::isfinite(beta[d])) return CELES_EINVAL;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    // a thread owns both polarisations of a direction while 2 nmax complex coefficients fit in registers (lmax <= 3)
    const int pols = ctx->lmax <= 3 ? 2 : 1;
    const int nmax = ctx->nmax, rows = 2 * n_dir, gx = (rows / pols + celes::kFarThreads - 1) / celes::kFarThreads;
    // split the sphere sum so that the grid has about four CTAs per SM-slot pair, at least 4 tiles per CTA
    int splits = std::max(1, std::min((8 * ctx->sm_count + gx - 1) / gx, std::max(1, ctx->N / (4 * celes::kFarTile))));
    const int chunk = ((ctx->N + splits - 1) / splits + celes::kFarTile - 1) / celes::kFarTile * celes::kFarTile;
    splits = (ctx->N + chunk - 1) / chunk;
    Scratch sc(ctx);
    int rc = sc.reserve(Scratch::align(sizeof(double) * 2 * (size_t)n_dir) + Scratch::align(sizeof(double) * 3 * (size_t)n_dir) +
                        Scratch::align(sizeof(float2) * (size_t)rows * nmax) + Scratch::align(sizeof(float2) * (size_t)rows * splits), s);
    if (rc) return rc;
    double* d_ang = sc.take<double>(2 * (size_t)n_dir);
    double* d_dir = sc.take<double>(3 * (size_t)n_dir);
    float2* d_coef = sc.take<float2>((size_t)rows * nmax);
    float2* d_part = sc.take<float2>((size_t)rows * splits);
    if (!rc && (cudaMemcpyAsync(d_ang, alpha, sizeof(double) * n_dir, cudaMemcpyHostToDevice, s) != cudaSuccess ||
                cudaMemcpyAsync(d_ang + n_dir, beta, sizeof(double) * n_dir, cudaMemcpyHostToDevice, s) != cudaSuccess)) rc = CELES_ECUDA;
    if (!rc) {
        celes::far_field_coefficients_kernel<<<(n_dir + 127) / 128, 128, 0, s>>>(ctx->lmax, n_dir, d_ang, d_ang + n_dir, d_coef, d_dir);
        const float2* b = (const float2*)b_dev;
        dim3 grid(gx, splits);
        switch (ctx->lmax) {
            case 1: celes::far_field_kernel<6, 2><<<grid, celes::kFarThreads, 0, s>>>(ctx->N, chunk, rows, ctx->kpos, b, d_coef, d_dir, d_part); break;
            case 2: celes::far_field_kernel<16, 2><<<grid, celes::kFarThreads, 0, s>>>(ctx->N, chunk, rows, ctx->kpos, b, d_coef, d_dir, d_part); break;
            case 3: celes::far_field_kernel<30, 2><<<grid, celes::kFarThreads, 0, s>>>(ctx->N, chunk, rows, ctx->kpos, b, d_coef, d_dir, d_part); break;
            case 4: celes::far_field_kernel<48, 1><<<grid, celes::kFarThreads, 0, s>>>(ctx->N, chunk, rows, ctx->kpos, b, d_coef, d_dir, d_part); break;
            case 5: celes::far_field_kernel<70, 1><<<grid, celes::kFarThreads, 0, s>>>(ctx->N, chunk, rows, ctx->kpos, b, d_coef, d_dir, d_part); break;
            default: rc = CELES_EINVAL;
        }
        if (!rc) celes::far_field_reduce_kernel<<<(rows + 255) / 256, 256, 0, s>>>(rows, splits, d_part, (float2*)g_dev);
        if (!rc && cudaGetLastError() != cudaSuccess) rc = CELES_ECUDA;
    }
    return rc;
}

// The same far field from the static scratch: no cudaMalloc, no cudaFree, no host allocation (see celes.h).  The launch
// configuration is the one celes_far_field would use (so is the result, bit for bit) unless the split partial sums would
// not fit the array, in which case the sphere sum is cut into fewer splits.
int celes_far_field_noalloc(celes_ctx* ctx, const void* b_dev, int n_dir, const double* alpha, const double* beta,
                            void* g_dev, void* cuda_stream) {
    if (!ctx || !b_dev || !g_dev || n_dir < 1 || !alpha || !beta) return CELES_EINVAL;
    if (n_dir > CELES_FAR_FIELD_NOALLOC_MAX_DIR) return CELES_ELIMIT;
    if (ctx->far_static == nullptr || ctx->nmax > 70) return CELES_ECUDA;      // set-up could not resolve the array
    for (int d = 0; d < n_dir; ++d)
        if (!std::isfinite(alpha[d]) || !std::isfinite(beta[d])) return CELES_EINVAL;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const int pols = ctx->lmax <= 3 ? 2 : 1;
    const int rows = 2 * n_dir, gx = (rows / pols + celes::kFarThreads - 1) / celes::kFarThreads;
    int splits = std::max(1, std::min((8 * ctx->sm_count + gx - 1) / gx, std::max(1, ctx->N / (4 * celes::kFarTile))));
    splits = std::max(1, std::min(splits, (int)(kFarStaticPartCapacity / (size_t)rows)));      // the partial sums must fit
    const int chunk = ((ctx->N + splits - 1) / splits + celes::kFarTile - 1) / celes::kFarTile * celes::kFarTile;
    splits = (ctx->N + chunk - 1) / chunk;
    unsigned char* base = static_cast<unsigned char*>(ctx->far_static);
    double* d_ang = reinterpret_cast<double*>(base + kFarStaticAngOff);
    double* d_dir = reinterpret_cast<double*>(base + kFarStaticDirOff);
    float2* d_coef = reinterpret_cast<float2*>(base + kFarStaticCoefOff);
    float2* d_part = reinterpret_cast<float2*>(base + kFarStaticPartOff);
    // nothing in the array has to start at zero: the three kernels below write every entry they later read (angles,
    // unit vectors, all nmax coefficients of all rows, one partial sum per (split, row)), so the previous call's
    // contents are simply overwritten
    if (cudaMemcpyAsync(d_ang, alpha, sizeof(double) * n_dir, cudaMemcpyHostToDevice, s) != cudaSuccess ||
        cudaMemcpyAsync(d_ang + n_dir, beta, sizeof(double) * n_dir, cudaMemcpyHostToDevice, s) != cudaSuccess) return CELES_ECUDA;
    celes::far_field_coefficients_kernel<<<(n_dir + 127) / 128, 128, 0, s>>>(ctx->lmax, n_dir, d_ang, d_ang + n_dir, d_coef, d_dir);
    const float2* b = (const float2*)b_dev;
    dim3 grid(gx, splits);
    switch (ctx->lmax) {
        case 1: celes::far_field_kernel<6, 2><<<grid, celes::kFarThreads, 0, s>>>(ctx->N, chunk, rows, ctx->kpos, b, d_coef, d_dir, d_part); break;
        case 2: celes::far_field_kernel<16, 2><<<grid, celes::kFarThreads, 0, s>>>(ctx->N, chunk, rows, ctx->kpos, b, d_coef, d_dir, d_part); break;
        case 3: celes::far_field_kernel<30, 2><<<grid, celes::kFarThreads, 0, s>>>(ctx->N, chunk, rows, ctx->kpos, b, d_coef, d_dir, d_part); break;
        case 4: celes::far_field_kernel<48, 1><<<grid, celes::kFarThreads, 0, s>>>(ctx->N, chunk, rows, ctx->kpos, b, d_coef, d_dir, d_part); break;
        case 5: celes::far_field_kernel<70, 1><<<grid, celes::kFarThreads, 0, s>>>(ctx->N, chunk, rows, ctx->kpos, b, d_coef, d_dir, d_part); break;
        default: return CELES_EINVAL;
    }
    celes::far_field_reduce_kernel<<<(rows + 255) / 256, 256, 0, s>>>(rows, splits, d_part, (float2*)g_dev);
    return cudaGetLastError() == cudaSuccess ? CELES_OK : CELES_ECUDA;
}

int celes_plane_wave(celes_ctx* ctx, double alpha, double beta, int polarisation, double E0_re, double E0_im, void* a_in_dev,
                     void* cuda_stream) {
    if (!ctx || !a_in_dev || (polarisation != 1 && polarisation != 2)) return CELES_EINVAL;
    if (!std::isfinite(alpha) || !std::isfinite(beta) || !std::isfinite(E0_re) || !std::isfinite(E0_im)) return CELES_EINVAL;
    const long long total = (long long)ctx->N * ctx->nmax;
    celes::plane_wave_kernel<<<(unsigned)((total + 127) / 128), 128, 0, (cudaStream_t)cuda_stream>>>(
        ctx->N, ctx->lmax, ctx->kpos, alpha, beta, polarisation, make_double2(E0_re, E0_im), (float2*)a_in_dev);
    return cudaGetLastError() == cudaSuccess ? CELES_OK : CELES_ECUDA;
}

static int gaussian_beam_impl(celes_ctx* ctx, const celes_beam* beam, void* a_in_dev, void* cuda_stream) {
    if (!ctx || !beam || !a_in_dev) return CELES_EINVAL;
    const int n_beta = beam->n_beta > 0 ? beam->n_beta : 400;
    if (!(beam->waist > 0.0) || !std::isfinite(beam->waist) || n_beta > 100000) return CELES_EINVAL;
    for (int a = 0; a < 3; ++a) if (!std::isfinite(beam->center[a])) return CELES_EINVAL;
    if (!std::isfinite(beam->alpha_G) || !std::isfinite(beam->E0_re) || !std::isfinite(beam->E0_im)) return CELES_EINVAL;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    std::vector<double> sb, cb;
    std::vector<double2> cminus, cplus;
    celes::gaussian_beam_tables(ctx->lmax, n_beta, ctx->k, beam->waist, sb, cb, cminus, cplus);
    Scratch sc(ctx);
    int rc = sc.reserve(2 * Scratch::align(sizeof(double) * n_beta) + Scratch::align(sizeof(double2) * cminus.size()) +
                        Scratch::align(sizeof(double2) * cplus.size()), s);
    if (rc) return rc;
    double* d_sb = sc.take<double>(n_beta);
    double* d_cb = sc.take<double>(n_beta);
    double2* d_cm = sc.take<double2>(cminus.size());
    double2* d_cp = sc.take<double2>(cplus.size());
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
    return rc;
}

int celes_gaussian_beam(celes_ctx* ctx, const celes_beam* beam, void* a_in_dev, void* cuda_stream) {
    CELES_NOTHROW(gaussian_beam_impl(ctx, beam, a_in_dev, cuda_stream))
}

static int scattered_field_impl(celes_ctx* ctx, const void* b_dev, int n_pts, const double* pts_xyz, void* e_dev, void* cuda_stream) {
    if (!ctx || !b_dev || !e_dev || !pts_xyz || n_pts < 1) return CELES_EINVAL;
    for (long long t = 0; t < 3LL * n_pts; ++t) if (!std::isfinite(pts_xyz[t])) return CELES_EINVAL;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    std::vector<double> kp(3 * (size_t)n_pts);
    for (size_t t = 0; t < kp.size(); ++t) kp[t] = ctx->k * pts_xyz[t];
    Scratch sc(ctx);
    int rc = sc.reserve(Scratch::align(sizeof(double) * kp.size()), s);
    if (rc) return rc;
    double* d_pts = sc.take<double>(kp.size());
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
    return rc;
}

int celes_scattered_field(celes_ctx* ctx, const void* b_dev, int n_pts, const double* pts_xyz, void* e_dev, void* cuda_stream) {
    CELES_NOTHROW(scattered_field_impl(ctx, b_dev, n_pts, pts_xyz, e_dev, cuda_stream))
}

}  // extern "C"
