// block_inverse.cuh -- step 3 of the block-diagonal preconditioner ("P_j M_j = L_j U_j", partial pivoting):
// every block M_j is inverted on the device by a blocked, in-place Gauss-Jordan elimination with row pivoting, all
// blocks of the preconditioner side by side in the same launches (one panel launch + one update launch per round).
//
// Round r treats the panel of columns [c0, c1) = [32 r, 32 r + 32) of every block that still has such columns:
//
//   gj_panel_kernel   one CTA per block.  The n x w panel is eliminated column by column: pivot = largest modulus among
//                     the rows >= c0 + s (lowest index on ties), row interchange, scaling, rank-1 update of all other rows.
//                     In place, so the panel ends up holding the columns c0..c1 of the composite row transformation
//                     G_r (the identity elsewhere); src[i] says which row of the old matrix is row i after the round's
//                     interchanges.  The panel lives in shared memory when n w fits, else in the destination buffer.
//   gj_update_kernel  strips of 64 columns, walked in 64 x 64 tiles, of all other columns:  new[i][j] = (i in [c0,c1) ? 0 : old[src[i]][j])
//                     + sum_t G[i][c0+t] old[src[c0+t]][j]  -- a rank-32 complex update in packed FFMA2.
//
// Everything happens IN PLACE in the one buffer that is kept.  The panel kernel owns the panel's columns; an update CTA
// owns ALL rows of its 64 columns and walks them top to bottom, so a tile only ever needs (a) its own rows, not yet
// overwritten, (b) the pivot rows and (c) the rows an interchange moved below the panel -- at most 32 per round, listed by
// the panel kernel (`disp_rows`) -- and it gathers (b) and (c) into shared memory before it writes anything.  After the
// last round the buffer holds B = (P A)^{-1} = A^{-1} P^T with P the accumulated row permutation `net` (row i of P A is row
// net[i] of A): z = A^{-1} v = B (P v), i.e. block_gemv_kernel reads v through net (precond_kernels.cuh).
#pragma once
#include <cuda_runtime.h>

#include "packed_math.cuh"

namespace celes {

constexpr int kGjNb = 32;          // panel width
constexpr int kGjThreads = 512;    // threads of a panel CTA
constexpr int kGjTile = 64;        // tile edge of the update kernel (256 threads, 4 x 4 outputs each)

struct GjBlocks {                  // device tables of the blocks, shared by both kernels
    int nmax;
    const int* by_size;            // [G] block indices, largest first (the active blocks of a round are a prefix)
    const int* grp_offset;         // [G+1] sphere offsets: n_j = (grp_offset[j+1] - grp_offset[j]) nmax; row tables start at grp_offset[j] nmax
    const long long* blk_offset;   // [G] element offset of block j in either buffer
    float2* buf;                   // the blocks, column-major, back to back
    int* src_row;                  // [N nmax] row interchange table of the current round
    int* disp_count;               // [G] rows below the panel whose content an interchange replaced (<= kGjNb)
    int* disp_rows;                // [G][kGjNb] their positions
    int* net;                      // [N nmax] accumulated permutation
    int* info;                     // [G] 1 = singular (zero or non-finite pivot)
};

__device__ __forceinline__ float2 cmulf(float2 a, float2 b) {
    return make_float2(fmaf(a.x, b.x, -a.y * b.y), fmaf(a.x, b.y, a.y * b.x));
}

__global__ void __launch_bounds__(kGjThreads) gj_panel_kernel(GjBlocks B, int round, int src_capacity, long long panel_capacity) {
    extern __shared__ __align__(16) unsigned char gj_smem[];
    __shared__ float red_val[kGjThreads / 32];
    __shared__ int red_idx[kGjThreads / 32];
    __shared__ float2 prow[kGjNb];
    const int j = B.by_size[blockIdx.x];
    const int g0 = B.grp_offset[j], n = (B.grp_offset[j + 1] - g0) * B.nmax;
    const int c0 = round * kGjNb;
    if (c0 >= n) return;
    const int w = min(kGjNb, n - c0);
    float2* neu = B.buf + B.blk_offset[j];
    int* src = reinterpret_cast<int*>(gj_smem);
    const bool in_smem = (long long)n * w <= panel_capacity;
    float2* P = in_smem ? reinterpret_cast<float2*>(gj_smem + (size_t)src_capacity * sizeof(int)) : neu + (size_t)c0 * n;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (in_smem)
        for (int e = tid; e < n * w; e += kGjThreads) P[e] = neu[(size_t)c0 * n + e];  // column-major panel, leading dimension n
    for (int i = tid; i < n; i += kGjThreads) src[i] = i;
    if (tid == 0) B.disp_count[j] = 0;
    __syncthreads();
    for (int s = 0; s < w; ++s) {
        const int pr = c0 + s;
        float2* Ps = P + (size_t)s * n;
        // pivot: largest modulus among the rows >= pr, lowest index on ties
        float best = -1.0f;
        int bi = n;
        for (int i = pr + tid; i < n; i += kGjThreads) {
            const float2 v = Ps[i];
            const float m = fmaf(v.x, v.x, v.y * v.y);
            if (m > best || !(m == m)) { best = m; bi = i; if (!(m == m)) break; }
        }
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) {
            const float ob = __shfl_down_sync(0xffffffffu, best, off);
            const int oi = __shfl_down_sync(0xffffffffu, bi, off);
            if (!(ob == ob) || (best == best && (ob > best || (ob == best && oi < bi)))) { best = ob; bi = oi; }
        }
        if (lane == 0) { red_val[warp] = best; red_idx[warp] = bi; }
        __syncthreads();
        best = red_val[0]; bi = red_idx[0];
#pragma unroll
        for (int q = 1; q < kGjThreads / 32; ++q) {
            const float ob = red_val[q];
            const int oi = red_idx[q];
            if (!(ob == ob) || (best == best && (ob > best || (ob == best && oi < bi)))) { best = ob; bi = oi; }
        }
        if (!(best > 0.0f) || !(best <= 3.0e38f)) {                      // singular or non-finite block: give up on it
            if (tid == 0) B.info[j] = 1;
            return;
        }
        if (bi != pr) {                                                    // row interchange inside the panel
            if (tid < w) { float2* col = P + (size_t)tid * n; const float2 t = col[pr]; col[pr] = col[bi]; col[bi] = t; }
            if (tid == kGjNb) { const int t = src[pr]; src[pr] = src[bi]; src[bi] = t; }
        }
        __syncthreads();
        const float2 a = Ps[pr];
        const float d = 1.0f / fmaf(a.x, a.x, a.y * a.y);
        const float2 inv = make_float2(a.x * d, -a.y * d);
        if (tid < w) prow[tid] = tid == s ? inv : cmulf(P[(size_t)tid * n + pr], inv);
        __syncthreads();
        for (int i = tid; i < n; i += kGjThreads) {                        // rank-1 update of every other row, in place
            float2* x = P + i;
            if (i == pr) {
                for (int t = 0; t < w; ++t, x += n) *x = prow[t];
                continue;
            }
            const float2 f = Ps[i], nf = make_float2(-f.x, -f.y);
            Ps[i] = make_float2(0.f, 0.f);                                 // column s becomes -f / a = 0 - f prow[s]
            int t = 0;
            for (; t + 4 <= w; t += 4, x += 4 * n) {
                const float2 x0 = x[0], x1 = x[n], x2 = x[2 * n], x3 = x[3 * n];
                x[0] = cfma2(nf, prow[t], x0); x[n] = cfma2(nf, prow[t + 1], x1);
                x[2 * n] = cfma2(nf, prow[t + 2], x2); x[3 * n] = cfma2(nf, prow[t + 3], x3);
            }
            for (; t < w; ++t, x += n) *x = cfma2(nf, prow[t], *x);
        }
        __syncthreads();
    }
    if (in_smem)
        for (int e = tid; e < n * w; e += kGjThreads) neu[(size_t)c0 * n + e] = P[e];
    const size_t rowbase = (size_t)g0 * B.nmax;
    for (int i = tid; i < n; i += kGjThreads) {
        const int si = src[i];
        B.src_row[rowbase + i] = si;
        if (i >= c0 + w && si != i) B.disp_rows[(size_t)j * kGjNb + atomicAdd(&B.disp_count[j], 1)] = i;   // order is immaterial
        src[i] = round == 0 ? si : B.net[rowbase + si];                    // net_new[i] = net_old[src[i]]
    }
    __syncthreads();
    for (int i = tid; i < n; i += kGjThreads) B.net[rowbase + i] = src[i];
}

// strip_off [n_active + 1]: prefix sums of ceil(n_j / 64) over the blocks in by_size order.  One CTA per strip of 64
// columns: the pivot rows and the displaced rows of the strip are gathered once, BEFORE anything is written, then the CTA
// walks down the strip in 64 x 64 tiles in place, loading the next tile (old values of its own rows + the panel's rows)
// into registers while the current one is being multiplied.
__global__ void __launch_bounds__(256, 2) gj_update_kernel(GjBlocks B, int round, int n_active, const long long* __restrict__ strip_off) {
    __shared__ __align__(16) float2 As[kGjNb][kGjTile];      // G[i0 + row][c0 + t]
    __shared__ __align__(16) float2 Bs[kGjNb][kGjTile];      // old[src[c0 + t]][j0 + col]
    __shared__ float2 Ds[kGjNb][kGjTile];                    // old[src[disp[k]]][j0 + col]: rows an interchange moved below the panel                    // (3 x 16 KB: the static shared-memory limit)
    int lo = 0, hi = n_active;
    const long long bid = blockIdx.x;
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (strip_off[mid] <= bid) lo = mid; else hi = mid;
    }
    const int j = B.by_size[lo];
    const int g0 = B.grp_offset[j], n = (B.grp_offset[j + 1] - g0) * B.nmax;
    const int c0 = round * kGjNb;
    if (c0 >= n) return;
    const int c1 = min(n, c0 + kGjNb), w = c1 - c0;
    const int tdim = (n + kGjTile - 1) / kGjTile;
    const int j0 = (int)(bid - strip_off[lo]) * kGjTile;
    const int jend = min(n, j0 + kGjTile);
    if (j0 >= c0 && jend <= c1) return;                                    // every column of the strip is a panel column
    float2* neu = B.buf + B.blk_offset[j];
    const float2* old = neu;                                               // in place: see the header of this file
    const int* src = B.src_row + (size_t)g0 * B.nmax;
    const int ndisp = B.disp_count[j];
    const int* disp = B.disp_rows + (size_t)j * kGjNb;
    const int tid = threadIdx.x;
    const int tx = tid & 15, ty = tid >> 4;
    const float2 zero = make_float2(0.f, 0.f);
    for (int e = tid; e < kGjNb * kGjTile; e += 256) {
        const int t = e >> 6, col = j0 + (e & 63);
        Bs[t][e & 63] = (t < w && col < n) ? old[(size_t)col * n + src[c0 + t]] : zero;
        if (t < ndisp && col < n) Ds[t][e & 63] = old[(size_t)col * n + src[disp[t]]];
    }
    __syncthreads();                                                       // everything gathered before the first store
    float2 pa[8], pc[4][4];
    auto prefetch = [&](int tm) {
        const int i0 = tm * kGjTile;
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            const int e = tid + 256 * q, t = e >> 6, row = i0 + (e & 63);
            pa[q] = (t < w && row < n) ? neu[(size_t)(c0 + t) * n + row] : zero;
        }
        int srow[4];
#pragma unroll
        for (int a = 0; a < 4; ++a) {
            const int row = i0 + tx + 16 * a;                              // lanes walk down a column: coalesced
            // >= 0: the row itself (not yet overwritten: tiles are walked top to bottom); -1: zero (pivot row or outside);
            // <= -2: displaced row, slot -2 - srow of Ds
            srow[a] = (row >= n || (row >= c0 && row < c1)) ? -1 : row;
            if (row >= c1 && row < n && ndisp > 0 && src[row] != row)
                for (int k = 0; k < ndisp; ++k) if (disp[k] == row) srow[a] = -2 - k;
        }
#pragma unroll
        for (int b = 0; b < 4; ++b) {
            const int col = j0 + 4 * ty + b, cl = 4 * ty + b;
#pragma unroll
            for (int a = 0; a < 4; ++a)
                pc[a][b] = col >= n ? zero : (srow[a] >= 0 ? old[(size_t)col * n + srow[a]] : (srow[a] == -1 ? zero : Ds[-2 - srow[a]][cl]));
        }
    };
    prefetch(0);
    for (int tm = 0; tm < tdim; ++tm) {
        __syncthreads();                                                   // the previous tile is done with As (and Bs is there)
#pragma unroll
        for (int q = 0; q < 8; ++q) { const int e = tid + 256 * q; As[e >> 6][e & 63] = pa[q]; }
        float2 acc[4][4];
#pragma unroll
        for (int a = 0; a < 4; ++a)
#pragma unroll
            for (int b = 0; b < 4; ++b) acc[a][b] = pc[a][b];
        __syncthreads();
        if (tm + 1 < tdim) prefetch(tm + 1);
#pragma unroll 4
        for (int t = 0; t < kGjNb; ++t) {                                  // rows t >= w of As and Bs are zero
            const float4 b01 = *reinterpret_cast<const float4*>(&Bs[t][4 * ty]), b23 = *reinterpret_cast<const float4*>(&Bs[t][4 * ty + 2]);
            const float2 av[4] = {As[t][tx], As[t][tx + 16], As[t][tx + 32], As[t][tx + 48]};
            const float2 bv[4] = {make_float2(b01.x, b01.y), make_float2(b01.z, b01.w), make_float2(b23.x, b23.y), make_float2(b23.z, b23.w)};
#pragma unroll
            for (int a = 0; a < 4; ++a)
#pragma unroll
                for (int b = 0; b < 4; ++b) acc[a][b] = cfma2(av[a], bv[b], acc[a][b]);
        }
        const int i0 = tm * kGjTile;
#pragma unroll
        for (int b = 0; b < 4; ++b) {
            const int col = j0 + 4 * ty + b;
            if (col >= n || (col >= c0 && col < c1)) continue;
#pragma unroll
            for (int a = 0; a < 4; ++a) {
                const int row = i0 + tx + 16 * a;
                if (row < n) neu[(size_t)col * n + row] = acc[a][b];
            }
        }
    }
}

}  // namespace celes
