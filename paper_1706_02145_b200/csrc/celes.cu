// celes.cu -- C-ABI library of the B200-native CELES hot path (include/celes.h).
//
// Host side of the boundary: argument validation, context (device tables + work space) and the kernel launches of
// y = W b (eq. 6-7) and out = b - T (W b) (eq. 8-9); the FP32 peak probes.  The
// solvers live in solve.cu, the preconditioner in precond.cu, beam / far field / near field in fields.cu.
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

#include "ctx.h"
#include "coupling_kernel.cuh"
#include "translation_table.h"
#include "work_partition.h"

namespace {

using celes::kBlock;

template <int LMAX, int ROT, bool TAB, bool EXT>
int launch_coupling_tt(const celes_ctx* c, cudaStream_t s, int rb0, int rb1) {
    const size_t smem = celes::coupling_smem_bytes<LMAX>(c->etile);
    const int cta0 = c->h_cta_of_block_first[rb0], cta1 = c->h_cta_of_block_last[rb1];
    celes::coupling_kernel<LMAX, ROT, TAB, EXT><<<cta1 - cta0 + 1, kBlock, smem, s>>>(
        c->N, c->bs, c->etile, cta0, rb0, rb1, c->htab_desc, c->cta_begin, c->seg, c->kpos, c->bpm, c->ypart);
    return cudaGetLastError() == cudaSuccess ? CELES_OK : CELES_ECUDA;
}

// The dynamic shared-memory limit is an attribute of the kernel for the whole process, not of a context: raise it once
// to the device's opt-in maximum so that contexts with different emitter tiles never lower it for one another.
template <int LMAX, int ROT, bool TAB, bool EXT>
int prepare_coupling_tt(celes_ctx* c, int* ctas_per_sm) {
    const size_t smem = celes::coupling_smem_bytes<LMAX>(c->etile);
    c->coupling_smem = smem;
    int optin = 0;
    CU_TRY(cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, c->device));
    if (smem > (size_t)optin) return CELES_EINVAL;             // emitter tile too large for this lmax
    CU_TRY(cudaFuncSetAttribute(celes::coupling_kernel<LMAX, ROT, TAB, EXT>, cudaFuncAttributeMaxDynamicSharedMemorySize, optin));
    CU_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(ctas_per_sm, celes::coupling_kernel<LMAX, ROT, TAB, EXT>, kBlock, smem));
    return CELES_OK;
}

// the table look-up and the extended range mode exist for the default (packed rotated) body only
template <int LMAX, int ROT>
int launch_coupling_t(const celes_ctx* c, cudaStream_t s, int rb0, int rb1) {
    if constexpr (ROT == celes::kRotated) {
        if (c->htab) return launch_coupling_tt<LMAX, ROT, true, false>(c, s, rb0, rb1);
        if (c->extended_range) return launch_coupling_tt<LMAX, ROT, false, true>(c, s, rb0, rb1);
    }
    return launch_coupling_tt<LMAX, ROT, false, false>(c, s, rb0, rb1);
}

template <int LMAX, int ROT>
int prepare_coupling_t(celes_ctx* c, int* ctas_per_sm) {
    if constexpr (ROT == celes::kRotated) {
        if (c->htab) return prepare_coupling_tt<LMAX, ROT, true, false>(c, ctas_per_sm);
        if (c->extended_range) return prepare_coupling_tt<LMAX, ROT, false, true>(c, ctas_per_sm);
    }
    return prepare_coupling_tt<LMAX, ROT, false, false>(c, ctas_per_sm);
}

#define CELES_DISPATCH(fn, ...)                                                            \
    switch (c->lmax * 2 + c->variant) {                                                    \
        case 2: return fn<1, 0>(__VA_ARGS__); case 3: return fn<1, 1>(__VA_ARGS__);        \
        case 4: return fn<2, 0>(__VA_ARGS__); case 5: return fn<2, 1>(__VA_ARGS__);        \
        case 6: return fn<3, 0>(__VA_ARGS__); case 7: return fn<3, 1>(__VA_ARGS__);        \
        case 8: return fn<4, 0>(__VA_ARGS__); case 9: return fn<4, 1>(__VA_ARGS__);        \
        case 10: return fn<5, 0>(__VA_ARGS__);   /* lmax = 5: packed rotated body only */  \
    }                                                                                      \
    return CELES_EINVAL

int launch_coupling(const celes_ctx* c, cudaStream_t s, int rb0, int rb1) { CELES_DISPATCH(launch_coupling_t, c, s, rb0, rb1); }
int prepare_coupling(celes_ctx* c, int* ctas_per_sm) { CELES_DISPATCH(prepare_coupling_t, c, ctas_per_sm); }

// y = W b (tdiag == nullptr) or out = b - T (W b): pack -> coupling -> finalize, all on stream s.
}  // namespace

int celes::host::run_matvec(celes_ctx* c, const float2* b, float2* out, bool system, cudaStream_t s, int row_begin,
                            int row_end) {
    if (row_begin < 0 || row_end > c->N || row_begin >= row_end) return CELES_EINVAL;
    const int H = c->nmax / 2;
    const long long nh = (long long)c->N * H;
    const int tb = 256;
    const unsigned gb = (unsigned)((nh + tb - 1) / tb);                      // every emitter's b is needed
    const unsigned gf = (unsigned)(((long long)(row_end - row_begin) * H + tb - 1) / tb);
    if (c->variant == celes::kRotated) celes::pack_kernel<celes::kRotated><<<gb, tb, 0, s>>>(c->N, H, b, c->bpm);
    else celes::pack_kernel<celes::kDirect><<<gb, tb, 0, s>>>(c->N, H, b, c->bpm);
    if (cudaGetLastError() != cudaSuccess) return CELES_ECUDA;
    int rc = launch_coupling(c, s, row_begin / c->bs, (row_end - 1) / c->bs);
    if (rc) return rc;
    const float2* td = system ? c->tdiag : nullptr;
    if (c->variant == celes::kRotated)
        celes::finalize_kernel<celes::kRotated><<<gf, tb, 0, s>>>(row_begin, row_end, H, c->bs, c->slot_begin, c->ypart, td, b, out);
    else
        celes::finalize_kernel<celes::kDirect><<<gf, tb, 0, s>>>(row_begin, row_end, H, c->bs, c->slot_begin, c->ypart, td, b, out);
    return cudaGetLastError() == cudaSuccess ? CELES_OK : CELES_ECUDA;
}

// Spheres must be disjoint ((A.5) needs |r| < |d|).  Uniform grid of cell edge 2 Rmax: every
// sphere is compared with the spheres of the 27 cells around it.  O(N log N).
namespace {

using celes::host::run_matvec;

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

void free_ctx(celes_ctx* c) {
    if (!c) return;
    celes::host::free_precond(c);
    celes::host::free_krylov(c);
    cudaFree(c->cta_begin); cudaFree(c->seg); cudaFree(c->slot_begin);
    cudaFree(c->kpos); cudaFree(c->tdiag); cudaFree(c->bpm); cudaFree(c->ypart); cudaFree(c->htab); cudaFree(c->host_in); cudaFree(c->host_out); cudaFree(c->scratch);
    delete c;
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
        case CELES_ELIMIT: return "size beyond the fixed capacity of a no-allocation entry point";
    }
    return "unknown error code";
}

static int translation_table_impl(int lmax, double* a5_re, double* b5_im) {
    if (lmax < CELES_LMAX_MIN || lmax > CELES_LMAX_MAX || !a5_re || !b5_im) return CELES_EINVAL;
    std::vector<double> a, b;
    if (!celes::build_translation_table(lmax, a, b)) return CELES_EINVAL;
    std::memcpy(a5_re, a.data(), sizeof(double) * a.size());
    std::memcpy(b5_im, b.data(), sizeof(double) * b.size());
    return CELES_OK;
}

int celes_translation_table(int lmax, double* a5_re, double* b5_im) { CELES_NOTHROW(translation_table_impl(lmax, a5_re, b5_im)) }

// the context under construction: released on every exit but the successful one (exceptions included)
struct CtxHolder {
    celes_ctx* c = nullptr;
    ~CtxHolder() { free_ctx(c); }
};

static int setup_impl(celes_ctx** out, int N, int lmax, const double* pos_xyz, const double* radii, const double* mie_q,
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
    if (opt && (opt->emitter_tile < 0 || opt->emitter_splits < 0 || opt->emitter_tile > 128 || opt->levels < 0)) return CELES_EINVAL;
    if (opt && (opt->translation < 0 || opt->translation > CELES_TRANSLATION_DIRECT)) return CELES_EINVAL;
    if (lmax > 4 && opt && opt->translation != CELES_TRANSLATION_ROTATED) return CELES_EINVAL;   // one body at lmax = 5
    const bool table = opt && opt->hankel == CELES_HANKEL_TABLE;
    if (opt && (opt->range < CELES_RANGE_AUTO || opt->range > CELES_RANGE_EXTENDED)) return CELES_EINVAL;
    if (opt && opt->range == CELES_RANGE_EXTENDED && (table || opt->translation != CELES_TRANSLATION_ROTATED)) return CELES_EINVAL;
    if (opt && opt->hankel != CELES_HANKEL_REGISTERS && opt->hankel != CELES_HANKEL_TABLE) return CELES_EINVAL;
    if (table && (opt->translation != CELES_TRANSLATION_ROTATED || !(opt->hankel_dr >= 0.0) || !std::isfinite(opt->hankel_dr)))
        return CELES_EINVAL;

    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { cudaGetLastError(); return CELES_ECUDA; }
    CtxHolder holder;
    celes_ctx* c = holder.c = new (std::nothrow) celes_ctx;
    if (!c) return CELES_ENOMEM;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    c->N = N; c->lmax = lmax; c->nmax = nmax; c->k = k;
    int rc = CELES_OK;
    auto fail = [&](int code) { return code; };                 // the holder releases the context
    if (cudaGetDevice(&c->device) != cudaSuccess) return fail(CELES_ECUDA);
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, c->device) != cudaSuccess) return fail(CELES_ECUDA);
    c->sm_count = prop.multiProcessorCount;
    // device address of the static scratch of celes_far_field_noalloc: looked up here, once per device, with this device current
    if (celes::host::far_static_scratch_address(c->device, &c->far_static) == CELES_ECUDA) return fail(CELES_ECUDA);
    // lmax = 5 spills ~0.5 KB per thread; a small tile leaves the L1 carve-out to those spills (measured: 17.8 ms with 8,
    // 19.2 ms with 32 at N = 1e4, profiles/r02d_other_kernels.md)
    c->etile = (opt && opt->emitter_tile > 0) ? opt->emitter_tile : (lmax >= 5 ? 8 : 32);
    c->variant = opt ? opt->translation : CELES_TRANSLATION_ROTATED;
    {   // extent of the cluster in units of 1/k: decides the range mode (celes.h: celes_options.range)
        double lo[3] = {pos_xyz[0], pos_xyz[1], pos_xyz[2]}, hi[3] = {pos_xyz[0], pos_xyz[1], pos_xyz[2]};
        for (int i = 0; i < N; ++i)
            for (int a = 0; a < 3; ++a) { lo[a] = std::min(lo[a], pos_xyz[3 * i + a]); hi[a] = std::max(hi[a], pos_xyz[3 * i + a]); }
        c->kd_max = k * std::sqrt((hi[0] - lo[0]) * (hi[0] - lo[0]) + (hi[1] - lo[1]) * (hi[1] - lo[1]) + (hi[2] - lo[2]) * (hi[2] - lo[2]));
        const int range = opt ? opt->range : CELES_RANGE_AUTO;
        const bool can = !table && c->variant == celes::kRotated;
        c->extended_range = can && (range == CELES_RANGE_EXTENDED || (range == CELES_RANGE_AUTO && c->kd_max > CELES_RANGE_AUTO_KD));
    }
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
    // work partition (work_partition.h): guided runs over the flattened (receiver block, emitter tile) grid, or the
    // caller's fixed number of emitter splits per receiver block
    c->fixed_splits = (opt && opt->emitter_splits > 0) ? opt->emitter_splits : 0;
    const int levels = (opt && opt->levels > 0) ? std::min(opt->levels, 16) : CELES_DEFAULT_LEVELS;
    celes::WorkPartition wp = celes::build_partition(N, kBlock, c->etile, c->sm_count * ctas_per_sm, levels, c->fixed_splits);
    c->bs = wp.bs; c->rblocks = wp.rblocks; c->n_cta = wp.n_cta; c->n_seg = (int)wp.seg.size();
    c->h_cta_of_block_first.assign(wp.rblocks, 0);
    c->h_cta_of_block_last.assign(wp.rblocks, 0);
    for (int cta = wp.n_cta - 1; cta >= 0; --cta)
        for (int t = wp.cta_begin[cta]; t < wp.cta_begin[cta + 1]; ++t) c->h_cta_of_block_first[wp.seg[t].rblock] = cta;
    for (int cta = 0; cta < wp.n_cta; ++cta)
        for (int t = wp.cta_begin[cta]; t < wp.cta_begin[cta + 1]; ++t) c->h_cta_of_block_last[wp.seg[t].rblock] = cta;

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
    SETUP_TRY(cudaMalloc(&c->ypart, sizeof(float2) * (size_t)c->n_seg * kBlock * nmax));
    SETUP_TRY(cudaMalloc(&c->cta_begin, sizeof(int) * wp.cta_begin.size()));
    SETUP_TRY(cudaMalloc(&c->seg, sizeof(int4) * wp.seg.size()));
    SETUP_TRY(cudaMalloc(&c->slot_begin, sizeof(int) * wp.slot_begin.size()));
    static_assert(sizeof(celes::Segment) == sizeof(int4), "Segment is read as int4 on the device");
    SETUP_TRY(cudaMemcpyAsync(c->cta_begin, wp.cta_begin.data(), sizeof(int) * wp.cta_begin.size(), cudaMemcpyHostToDevice, s));
    SETUP_TRY(cudaMemcpyAsync(c->seg, wp.seg.data(), sizeof(int4) * wp.seg.size(), cudaMemcpyHostToDevice, s));
    SETUP_TRY(cudaMemcpyAsync(c->slot_begin, wp.slot_begin.data(), sizeof(int) * wp.slot_begin.size(), cudaMemcpyHostToDevice, s));
    SETUP_TRY(cudaMemcpyAsync(c->kpos, kp.data(), sizeof(double) * kp.size(), cudaMemcpyHostToDevice, s));
    SETUP_TRY(cudaMemcpyAsync(c->tdiag, td.data(), sizeof(float2) * n, cudaMemcpyHostToDevice, s));
    SETUP_TRY(cudaStreamSynchronize(s));
#undef SETUP_TRY
    *out = c;
    holder.c = nullptr;
    return CELES_OK;
}

int celes_setup(celes_ctx** out, int N, int lmax, const double* pos_xyz, const double* radii, const double* mie_q,
                double k, const celes_options* opt, void* cuda_stream) {
    CELES_NOTHROW(setup_impl(out, N, lmax, pos_xyz, radii, mie_q, k, opt, cuda_stream))
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
    if (emitter_splits) *emitter_splits = ctx->fixed_splits;
    if (block_threads) *block_threads = kBlock;
    if (emitter_tile) *emitter_tile = ctx->etile;
    return CELES_OK;
}

#ifdef CELES_TRACE
int celes_debug_trace(unsigned long long* out) {
    return cudaMemcpyFromSymbol(out, celes::g_trace, sizeof(unsigned long long) * 3 * 8192) == cudaSuccess ? CELES_OK : CELES_ECUDA;
}
#endif

int celes_range_info(const celes_ctx* ctx, double* kd_max, int* extended) {
    if (!ctx) return CELES_EINVAL;
    if (kd_max) *kd_max = ctx->kd_max;
    if (extended) *extended = ctx->extended_range ? 1 : 0;
    return CELES_OK;
}

int celes_work_partition(const celes_ctx* ctx, int* ctas, int* segments, int* receivers_per_block) {
    if (!ctx) return CELES_EINVAL;
    if (ctas) *ctas = ctx->n_cta;
    if (segments) *segments = ctx->n_seg;
    if (receivers_per_block) *receivers_per_block = ctx->bs;
    return CELES_OK;
}

int celes_plan_work(int N, int emitter_tile, int resident_ctas, int levels, int emitter_splits, int* ctas, int* segments,
                    int* receivers_per_block, int* seg_out, int seg_capacity) {
    if (N < 1 || emitter_tile < 1 || resident_ctas < 1 || emitter_splits < 0 || levels < 0) return CELES_EINVAL;
    try {
        const celes::WorkPartition wp = celes::build_partition(N, kBlock, emitter_tile, resident_ctas,
                                                               levels > 0 ? levels : CELES_DEFAULT_LEVELS, emitter_splits);
        if (ctas) *ctas = wp.n_cta;
        if (segments) *segments = (int)wp.seg.size();
        if (receivers_per_block) *receivers_per_block = wp.bs;
        if (seg_out) {
            if (seg_capacity < (int)wp.seg.size()) return CELES_EINVAL;
            for (int cta = 0; cta < wp.n_cta; ++cta)
                for (int t = wp.cta_begin[cta]; t < wp.cta_begin[cta + 1]; ++t) {
                    const celes::Segment& sg = wp.seg[t];
                    int* o = seg_out + 5 * (size_t)t;
                    o[0] = cta; o[1] = sg.rblock; o[2] = sg.e_begin; o[3] = sg.e_end; o[4] = sg.slot;
                }
        }
    } catch (const std::bad_alloc&) {
        return CELES_ENOMEM;
    }
    return CELES_OK;
}

int celes_coupling_matvec_rows(celes_ctx* ctx, int row_begin, int row_end, const void* b_dev, void* y_rows_dev, void* cuda_stream) {
    if (!ctx || !b_dev || !y_rows_dev || b_dev == y_rows_dev) return CELES_EINVAL;
    return run_matvec(ctx, (const float2*)b_dev, (float2*)y_rows_dev, false, (cudaStream_t)cuda_stream, row_begin, row_end);
}

int celes_system_matvec_rows(celes_ctx* ctx, int row_begin, int row_end, const void* b_dev, void* out_rows_dev, void* cuda_stream) {
    if (!ctx || !b_dev || !out_rows_dev || b_dev == out_rows_dev) return CELES_EINVAL;
    return run_matvec(ctx, (const float2*)b_dev, (float2*)out_rows_dev, true, (cudaStream_t)cuda_stream, row_begin, row_end);
}

void celes_destroy(celes_ctx* ctx) { free_ctx(ctx); }

}  // extern "C"
