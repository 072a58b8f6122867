// solve.cu -- celes_solve: host-driven restarted GMRES and BiCGSTAB on M x = T a_in, every vector
// operation a device kernel (krylov_kernels.cuh), optional right preconditioning with the block-diagonal operator.
#include <cuda_runtime.h>
#include <cstdlib>
#include <cstdio>

#include <algorithm>
#include <chrono>
#include <cmath>
#include <complex>
#include <cstring>
#include <functional>
#include <vector>

#include "ctx.h"
#include "krylov_kernels.cuh"

using celes::host::precond_apply;
using celes::host::run_matvec;

void celes::host::free_krylov(celes_ctx* c) {
    cudaFree(c->V); cudaFree(c->rhs); cudaFree(c->tmp); cudaFree(c->partial); cudaFree(c->coef); cudaFree(c->hsum);
    if (c->hhost) cudaFreeHost(c->hhost);
    for (int q = 0; q < 2; ++q) if (c->kry_ev[q]) { cudaEventDestroy(c->kry_ev[q]); c->kry_ev[q] = nullptr; }
    c->V = nullptr; c->rhs = c->tmp = nullptr; c->partial = c->coef = c->hsum = nullptr; c->hhost = nullptr;
    c->kry_restart = 0;
}

namespace {

// Work space of the solvers, sized for `restart`.  All or nothing: a failed (re-)allocation releases everything and
// leaves kry_restart = 0, so a later call can never run on a half-allocated work space.
int ensure_krylov(celes_ctx* c, int restart) {
    if (c->V && c->kry_restart >= restart) return CELES_OK;
    celes::host::free_krylov(c);
    const size_t n = (size_t)c->N * c->nmax;
    c->dot_blocks = (int)std::min<size_t>((n + celes::kDotBlock - 1) / celes::kDotBlock, (size_t)c->sm_count * 4);
    cudaError_t e = cudaMalloc(&c->V, sizeof(float2) * n * (restart + 1));
    if (e == cudaSuccess) e = cudaMalloc(&c->rhs, sizeof(float2) * n);
    if (e == cudaSuccess) e = cudaMalloc(&c->tmp, sizeof(float2) * n);
    if (e == cudaSuccess) e = cudaMalloc(&c->partial, sizeof(double2) * c->dot_blocks * (restart + 1));
    if (e == cudaSuccess) e = cudaMalloc(&c->coef, sizeof(double2) * (restart + 2));
    if (e == cudaSuccess) e = cudaMalloc(&c->hsum, sizeof(double2) * 2 * (restart + 2));
    if (e == cudaSuccess) e = cudaMallocHost(&c->hhost, sizeof(double2) * 3 * (restart + 2));
    for (int q = 0; q < 2 && e == cudaSuccess; ++q) e = cudaEventCreateWithFlags(&c->kry_ev[q], cudaEventDisableTiming);
    if (e != cudaSuccess) {
        celes::host::free_krylov(c);
        cudaGetLastError();
        return e == cudaErrorMemoryAllocation ? CELES_ENOMEM : CELES_ECUDA;
    }
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
static int solve_impl(celes_ctx* ctx, const void* a_in_dev, void* x_dev, const celes_solve_opts* o, celes_solve_info* info,
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
    if (info) std::memset(info, 0, sizeof(*info));
    int rc = ensure_krylov(ctx, method == CELES_BICGSTAB ? std::max(restart, 8) : restart);
    if (rc) return rc;
    const long long n = (long long)ctx->N * ctx->nmax;
    const int eb = (int)std::min<long long>((n + 255) / 256, (long long)ctx->sm_count * 8);
    float2* x = (float2*)x_dev;
    float2* V = ctx->V;
    typedef std::complex<double> cd;

    int iterations = 0, matvecs = 0, n_hist = 0, converged = 0;
    double rel = 0.0;
    auto push_hist = [&](double v) { if (info && n_hist < CELES_MAX_HISTORY) info->history[n_hist++] = v; };
    // diagnostic (CELES_DEBUG set): host time at which every Hessenberg column arrived; finish() prints how the gaps between
    // them are distributed -- a few long gaps mean host / driver hiccups, uniformly longer ones a slower GPU
    const bool dbg_gaps = std::getenv("CELES_DEBUG") != nullptr;
    constexpr int kMaxStamps = 4096;
    double stamp[kMaxStamps];
    int n_stamp = 0;
    auto finish = [&](int code) {
        if (dbg_gaps && n_stamp > 3) {
            double gap[kMaxStamps];
            for (int t = 1; t < n_stamp; ++t) gap[t - 1] = stamp[t] - stamp[t - 1];
            const int ng = n_stamp - 1;
            int at = 0;
            for (int t = 1; t < ng; ++t) if (gap[t] > gap[at]) at = t;          // which arrival the longest wait preceded
            std::sort(gap, gap + ng);
            const double med = gap[ng / 2];
            double excess = 0.0; int n_long = 0;
            for (int t = 0; t < ng; ++t) if (gap[t] > 1.5 * med) { excess += gap[t] - med; ++n_long; }
            std::fprintf(stderr, "celes_solve gaps ms: n %d | median %.3f | p90 %.3f | max %.3f %.3f %.3f | longest before arrival %d | %d gaps > 1.5 median hold %.2f ms of excess | total %.1f\n",
                         ng, 1e3 * med, 1e3 * gap[(int)(0.9 * ng)], 1e3 * gap[ng - 1], 1e3 * gap[ng - 2], 1e3 * gap[ng - 3], at + 1, n_long, 1e3 * excess,
                         1e3 * (stamp[n_stamp - 1] - stamp[0]));
        }
        if (info) {
            info->iterations = iterations; info->matvecs = matvecs; info->converged = converged;
            info->rel_residual = rel; info->n_history = n_hist;
            info->seconds = std::chrono::duration<double>(std::chrono::steady_clock::now() - t_start).count();
        }
        return code;
    };

#define SOLVE_TRY(expr)                                                                          \
    do {                                                                                         \
        cudaError_t e_ = (expr);                                                                 \
        if (e_ != cudaSuccess) return finish(e_ == cudaErrorMemoryAllocation ? CELES_ENOMEM : CELES_ECUDA); \
    } while (0)
    // rhs = T a_in (eq. 8)
    celes::tapply_kernel<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(n, ctx->tdiag, (const float2*)a_in_dev, ctx->rhs);
    double fnorm = 0.0;
    rc = device_norm(ctx, n, ctx->rhs, &fnorm, s);
    if (rc) return finish(rc);
    if (fnorm == 0.0) {                       // zero right-hand side: x = 0
        SOLVE_TRY(cudaMemsetAsync(x, 0, sizeof(float2) * n, s));
        SOLVE_TRY(cudaStreamSynchronize(s));
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
            SOLVE_TRY(cudaMemsetAsync(hsum, 0, sizeof(double2) * (jc + 2), s));
            for (int pass = 0; pass < 2; ++pass) {
                r2 = device_dots(ctx, n, jc + 1, V, w, ctx->coef, hsum, s);
                if (r2) return r2;
                r2 = device_axpys(ctx, n, jc + 1, -1.0, ctx->coef, V, w, s);
                if (r2) return r2;
            }
            r2 = device_dots(ctx, n, 1, w, w, hsum + (jc + 1), nullptr, s);
            if (r2) return r2;
            celes::scale_by_inv_norm_kernel<<<eb, 256, 0, s>>>(n, hsum + (jc + 1), w, w);
            SOLVE_TRY(cudaMemcpyAsync(ctx->hhost + (size_t)(jc & 1) * hs, hsum, sizeof(double2) * (jc + 2), cudaMemcpyDeviceToHost, s));
            SOLVE_TRY(cudaEventRecord(ctx->kry_ev[jc & 1], s));
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
            SOLVE_TRY(cudaEventSynchronize(ctx->kry_ev[j & 1]));
            if (dbg_gaps && n_stamp < kMaxStamps) stamp[n_stamp++] = std::chrono::duration<double>(std::chrono::steady_clock::now() - t_start).count();
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
        SOLVE_TRY(cudaMemcpyAsync(ctx->coef, hup, sizeof(double2) * j, cudaMemcpyHostToDevice, s));
        if (j > 0 && pc) {                                     // x += P^{-1} (V y)
            SOLVE_TRY(cudaMemsetAsync(ctx->tmp, 0, sizeof(float2) * n, s));
            rc = device_axpys(ctx, n, j, 1.0, ctx->coef, V, ctx->tmp, s);
            if (rc) return finish(rc);
            rc = precond_apply(ctx, ctx->tmp, ctx->pc_tmp, s);
            if (rc) return finish(rc);
            celes::add_kernel<<<eb, 256, 0, s>>>(n, ctx->pc_tmp, x);
        } else if (j > 0) {
            rc = device_axpys(ctx, n, j, 1.0, ctx->coef, V, x, s);
            if (rc) return finish(rc);
        }
        SOLVE_TRY(cudaStreamSynchronize(s));      // hhost is reused by the next cycle
    }
#undef SOLVE_TRY
}

int celes_solve(celes_ctx* ctx, const void* a_in_dev, void* x_dev, const celes_solve_opts* o, celes_solve_info* info,
                void* cuda_stream) {
    CELES_NOTHROW(solve_impl(ctx, a_in_dev, x_dev, o, info, cuda_stream))
}

}  // extern "C"
