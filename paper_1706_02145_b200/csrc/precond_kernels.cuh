// precond_kernels.cuh -- device kernels of the block-diagonal preconditioner (section 3.2.1).
//
//   assemble_blocks_kernel  step 2: the dense blocks M_j = 1 - T W restricted to the spheres of subset G_j, from the
//                           addition theorem (A.6)-(A.8) term by term with the run-time a5/b5 table --
//                           an evaluation of W that is independent of the generated pair bodies
//   (block_inverse.cuh)     step 3: pivoted elimination of every block, all blocks in the same launches
//   block_gemv_kernel       step 4: z = blockdiag(M_j^{-1}) v.  The blocks hold the explicit inverses (obtained from
//                           the pivoted elimination of step 3), so that applying the preconditioner is one batched,
//                           HBM-bound matrix-vector product instead of per-block triangular solves.
#pragma once
#include <cuda_runtime.h>

namespace celes {

constexpr int kAsmThreads = 96;     // >= nmax of every supported lmax (70 at lmax = 5)
constexpr int kGemvRows = 128;      // rows of a block handled by one CTA of block_gemv_kernel
constexpr int kGemvChunk = 1024;    // block_gemv_chunked_kernel: columns whose x values are staged at a time (8 KB)
constexpr int kGemvChunkedFrom = 1536;   // largest block above this many rows: the chunked kernel (measured crossover)

// One CTA per ordered pair (a, b) of spheres of one subset; thread t < nmax fills column n' = t of the nmax x nmax
// block  M^{ab} = delta_ab 1 - T^a W^{ab}  inside the column-major n_j x n_j matrix of the subset.
//   pair_offset [n_groups+1]: prefix sums of N_j^2;  blk_offset [n_groups]: start (in elements) of M_j in blocks;
//   a5, b5 [H][H][P]: Re a5(l',m'|l,m|p), Im b5(l',m'|l,m|p), receiver index first (celes_translation_table layout).
template <int LMAX>
__global__ void __launch_bounds__(kAsmThreads) assemble_blocks_kernel(
    int n_groups, const long long* __restrict__ pair_offset, const int* __restrict__ grp_offset,
    const int* __restrict__ order, const long long* __restrict__ blk_offset, const double* __restrict__ kpos,
    const float2* __restrict__ tdiag, const float* __restrict__ a5, const float* __restrict__ b5,
    float2* __restrict__ blocks) {
    constexpr int H = LMAX * (LMAX + 2), NMAX = 2 * H, P = 2 * LMAX + 1;
    __shared__ float2 G[P][P];          // G[p][nu] = h_p(kd) P_p^nu(cos theta)
    __shared__ float2 E[P];             // e^{i nu phi}
    __shared__ float2 tile[NMAX][NMAX + 1];   // tile[n'][n]: the block, staged so that it leaves in runs of consecutive rows
    // subset of this pair: binary search in the prefix sums
    const long long bid = blockIdx.x;
    int lo = 0, hi = n_groups;
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (pair_offset[mid] <= bid) lo = mid; else hi = mid;
    }
    const int j = lo, g0 = grp_offset[j], nj = grp_offset[j + 1] - g0;
    const int local = (int)(bid - pair_offset[j]);
    const int a = local / nj, b = local - a * nj;
    const int i = order[g0 + a], ip = order[g0 + b];
    const size_t ld = (size_t)nj * NMAX;
    float2* Mj = blocks + blk_offset[j];
    const int t = threadIdx.x;
    float2* out = Mj + (size_t)(a * NMAX) + (size_t)(b * NMAX) * ld;   // element (n, n') at out[n + n' ld]
    if (a == b) {                                           // W^{ii} = 0: identity block
        for (int e = t; e < NMAX * NMAX; e += kAsmThreads) {
            const int c = e / NMAX, n = e - c * NMAX;
            out[(size_t)c * ld + n] = make_float2(n == c ? 1.0f : 0.0f, 0.0f);
        }
        return;
    }
    // geometry of d = r_i - r_i'; subtraction in FP64 as in the coupling kernel
    const float dx = (float)(kpos[3 * i] - kpos[3 * ip]), dy = (float)(kpos[3 * i + 1] - kpos[3 * ip + 1]),
                dz = (float)(kpos[3 * i + 2] - kpos[3 * ip + 2]);
    const float rho2 = fmaf(dx, dx, dy * dy), r2 = fmaf(dz, dz, rho2);
    const float rinv = rsqrtf(r2), x = r2 * rinv, ct = dz * rinv;
    const bool on_axis = rho2 < 1e-12f * r2;
    const float rhoinv = on_axis ? 0.0f : rsqrtf(rho2);
    const float cph = on_axis ? 1.0f : dx * rhoinv, sph = on_axis ? 0.0f : dy * rhoinv;
    const float st = rho2 * rhoinv * rinv;
    if (t < P) {                                            // thread nu = t: column nu of the Legendre triangle
        const int nu = t;
        float sx, cx;
        sincosf(x, &sx, &cx);
        float hr[P], hi_[P];
        hr[0] = sx * rinv; hi_[0] = -cx * rinv;
        hr[1] = fmaf(sx, rinv, -cx) * rinv; hi_[1] = -fmaf(cx, rinv, sx) * rinv;
        for (int p = 1; p + 1 < P; ++p) {
            const float f = (float)(2 * p + 1) * rinv;
            hr[p + 1] = fmaf(f, hr[p], -hr[p - 1]);
            hi_[p + 1] = fmaf(f, hi_[p], -hi_[p - 1]);
        }
        // normalised associated Legendre functions without Condon-Shortley phase: P_nu^nu, then upward in p
        float pmm = 0.70710678118654752f;
        for (int mu = 1; mu <= nu; ++mu) pmm *= sqrtf((2.0f * mu + 1.0f) / (2.0f * mu)) * st;
        float pm2 = 0.0f, pm1 = pmm;
        for (int p = 0; p < P; ++p) {
            float val = 0.0f;
            if (p == nu) val = pmm;
            else if (p > nu) {
                const float fp = (float)p, fn = (float)nu;
                const float c1 = sqrtf((4.0f * fp * fp - 1.0f) / (fp * fp - fn * fn));
                const float c2 = sqrtf(((fp - 1.0f) * (fp - 1.0f) - fn * fn) / (4.0f * (fp - 1.0f) * (fp - 1.0f) - 1.0f));
                val = c1 * (ct * pm1 - c2 * pm2);
                pm2 = pm1; pm1 = val;
            }
            G[p][nu] = make_float2(hr[p] * val, hi_[p] * val);
        }
        float cr = 1.0f, ci = 0.0f;                          // e^{i nu phi}
        for (int mu = 0; mu < nu; ++mu) { const float tr = cr * cph - ci * sph; ci = cr * sph + ci * cph; cr = tr; }
        E[nu] = make_float2(cr, ci);
    }
    __syncthreads();
    if (t < NMAX) {
    const int taup = t / H, cq = t - taup * H;              // emitter n' = (tau', l', m')
    int lp = 1;
    while ((lp + 1) * (lp + 1) - 1 <= cq) ++lp;
    const int mp = cq - (lp * lp - 1) - lp;
    float2* col = tile[t];
    const float2* ta = tdiag + (size_t)i * NMAX;
    int rq = 0;
    for (int l = 1; l <= LMAX; ++l)
        for (int m = -l; m <= l; ++m, ++rq) {
            const int mu = mp - m, nu = mu < 0 ? -mu : mu;
            const float* ca = a5 + ((size_t)rq * H + cq) * P;
            const float* cb = b5 + ((size_t)rq * H + cq) * P;
            float ar = 0.f, ai = 0.f, br = 0.f, bi = 0.f;     // sum_p a5 G,  sum_p b5'' G
            const int p0 = max(abs(l - lp), nu);
            for (int p = p0; p <= l + lp; ++p) {
                const float2 g = G[p][nu];
                ar = fmaf(ca[p], g.x, ar); ai = fmaf(ca[p], g.y, ai);
                br = fmaf(cb[p], g.x, br); bi = fmaf(cb[p], g.y, bi);
            }
            // times e^{i mu phi}; b5 = i b5''
            const float er = E[nu].x, ei = mu < 0 ? -E[nu].y : E[nu].y;
            const float2 A = make_float2(ar * er - ai * ei, ar * ei + ai * er);
            const float2 B = make_float2(-(br * ei + bi * er), br * er - bi * ei);
            for (int tau = 0; tau < 2; ++tau) {
                const float2 w = tau == taup ? A : B;
                const float2 q = ta[tau * H + rq];
                col[tau * H + rq] = make_float2(-(q.x * w.x - q.y * w.y), -(q.x * w.y + q.y * w.x));   // a != b: no delta
            }
        }
    }
    __syncthreads();
    for (int e = t; e < NMAX * NMAX; e += kAsmThreads) {   // consecutive threads, consecutive rows of one column
        const int c = e / NMAX, n = e - c * NMAX;
        out[(size_t)c * ld + n] = tile[c][n];
    }
}

// z = blockdiag(Minv_j) v.  CTA c handles rows [row0, row0 + kGemvRows) of subset cta_group[c]; one thread per row,
// the subset's slice of v gathered into shared memory (broadcast reads), the matrix read once, coalesced along rows.
// The stored block is B_j = M_j^{-1} P_j^T with P_j the row permutation of the pivoted elimination (block_inverse.cuh):
// M_j^{-1} v = B_j (P_j v), so column c of B_j meets element perm[c] of the subset's slice.
__global__ void __launch_bounds__(kGemvRows) block_gemv_kernel(
    int nmax, const int* __restrict__ cta_group, const int* __restrict__ cta_row0, const int* __restrict__ grp_offset,
    const int* __restrict__ order, const long long* __restrict__ blk_offset, const int* __restrict__ perm,
    const float2* __restrict__ blocks, const float2* __restrict__ v, float2* __restrict__ z) {
    extern __shared__ float2 xs[];
    const int j = cta_group[blockIdx.x], row0 = cta_row0[blockIdx.x];
    const int g0 = grp_offset[j], nj = grp_offset[j + 1] - g0, n = nj * nmax;
    const int* pj = perm + (size_t)g0 * nmax;
    for (int c = threadIdx.x; c < n; c += kGemvRows) {
        const int pc = pj[c], s = pc / nmax;
        xs[c] = v[(size_t)order[g0 + s] * nmax + (pc - s * nmax)];
    }
    __syncthreads();
    const int r = row0 + threadIdx.x;
    if (r >= n) return;
    const float2* A = blocks + blk_offset[j] + r;
    float ar0 = 0.f, ai0 = 0.f, ar1 = 0.f, ai1 = 0.f;
    int c = 0;
    for (; c + 1 < n; c += 2) {
        const float2 m0 = A[(size_t)c * n], m1 = A[(size_t)(c + 1) * n];
        const float2 x0 = xs[c], x1 = xs[c + 1];
        ar0 = fmaf(m0.x, x0.x, ar0); ar0 = fmaf(-m0.y, x0.y, ar0); ai0 = fmaf(m0.x, x0.y, ai0); ai0 = fmaf(m0.y, x0.x, ai0);
        ar1 = fmaf(m1.x, x1.x, ar1); ar1 = fmaf(-m1.y, x1.y, ar1); ai1 = fmaf(m1.x, x1.y, ai1); ai1 = fmaf(m1.y, x1.x, ai1);
    }
    if (c < n) {
        const float2 m0 = A[(size_t)c * n], x0 = xs[c];
        ar0 = fmaf(m0.x, x0.x, ar0); ar0 = fmaf(-m0.y, x0.y, ar0); ai0 = fmaf(m0.x, x0.y, ai0); ai0 = fmaf(m0.y, x0.x, ai0);
    }
    const int s = r / nmax;
    z[(size_t)order[g0 + s] * nmax + (r - s * nmax)] = make_float2(ar0 + ar1, ai0 + ai1);
}

// The same product for TALL blocks.  block_gemv_kernel keeps the whole x slice of its block in shared memory, which caps the
// resident CTAs once a block has a few thousand rows (22 KB per CTA at 2736 rows: 9 CTAs per SM instead of 16) and with
// them the loads in flight; here x streams through a fixed 8 KB chunk, so occupancy does not depend on the block.
// Measured (profiles/r02r_block_gemv_tall_blocks.md): 0.64 -> 0.93 of the HBM copy bandwidth at 1980 rows, but 0.92 -> 0.70 at
// 672 rows (two barriers per chunk and no long uninterrupted column loop), hence the dispatch by the largest block's size.
__global__ void __launch_bounds__(kGemvRows) block_gemv_chunked_kernel(
    int nmax, const int* __restrict__ cta_group, const int* __restrict__ cta_row0, const int* __restrict__ grp_offset,
    const int* __restrict__ order, const long long* __restrict__ blk_offset, const int* __restrict__ perm,
    const float2* __restrict__ blocks, const float2* __restrict__ v, float2* __restrict__ z) {
    __shared__ float2 xs[kGemvChunk];
    const int j = cta_group[blockIdx.x], row0 = cta_row0[blockIdx.x];
    const int g0 = grp_offset[j], nj = grp_offset[j + 1] - g0, n = nj * nmax;
    const int* pj = perm + (size_t)g0 * nmax;
    const int r = row0 + threadIdx.x;
    const bool active = r < n;
    const float2* A = blocks + blk_offset[j] + (active ? r : 0);
    float ar0 = 0.f, ai0 = 0.f, ar1 = 0.f, ai1 = 0.f;
    for (int c0 = 0; c0 < n; c0 += kGemvChunk) {
        const int nc = min(kGemvChunk, n - c0);
        __syncthreads();                                               // the previous chunk is consumed
        for (int c = threadIdx.x; c < nc; c += kGemvRows) {
            const int pc = pj[c0 + c], s = pc / nmax;
            xs[c] = v[(size_t)order[g0 + s] * nmax + (pc - s * nmax)];
        }
        __syncthreads();
        if (active) {
            const float2* Ac = A + (size_t)c0 * n;
            int c = 0;
            for (; c + 1 < nc; c += 2) {
                const float2 m0 = Ac[(size_t)c * n], m1 = Ac[(size_t)(c + 1) * n];
                const float2 x0 = xs[c], x1 = xs[c + 1];
                ar0 = fmaf(m0.x, x0.x, ar0); ar0 = fmaf(-m0.y, x0.y, ar0); ai0 = fmaf(m0.x, x0.y, ai0); ai0 = fmaf(m0.y, x0.x, ai0);
                ar1 = fmaf(m1.x, x1.x, ar1); ar1 = fmaf(-m1.y, x1.y, ar1); ai1 = fmaf(m1.x, x1.y, ai1); ai1 = fmaf(m1.y, x1.x, ai1);
            }
            if (c < nc) {
                const float2 m0 = Ac[(size_t)c * n], x0 = xs[c];
                ar0 = fmaf(m0.x, x0.x, ar0); ar0 = fmaf(-m0.y, x0.y, ar0); ai0 = fmaf(m0.x, x0.y, ai0); ai0 = fmaf(m0.y, x0.x, ai0);
            }
        }
    }
    if (!active) return;
    const int s = r / nmax;
    z[(size_t)order[g0 + s] * nmax + (r - s * nmax)] = make_float2(ar0 + ar1, ai0 + ai1);
}

}  // namespace celes
