// pair_math.cuh -- per-pair arithmetic of the direct coupling kernel (steps H2-H7 of DESIGN.md).
//
// For the ordered pair (receiver i, emitter i') with d = r_i - r_i' (eq. 7) this evaluates
// h_p^(1)(kd), P_p^nu(cos theta_d), e^{i nu phi_d} in registers and applies the 2x2 tau-block translation
// (A.6)-(A.8), to the emitter's coefficients.  The contraction itself is generated code
// (generated/coupling_body_lmax*.inc, written by gen_coupling_body.py).
#pragma once

#include "hankel_table.h"
#include "variants.h"
#include "packed_math.cuh"

template <int LMAX>
struct PairBody;   // specialised by the generated files

#include "generated/coupling_body_lmax1.inc"
#include "generated/coupling_body_lmax2.inc"
#include "generated/coupling_body_lmax3.inc"
#include "generated/coupling_body_lmax4.inc"

template <int LMAX>
struct PairBodyPk;    // packed (FFMA2) rotate / axial-translate / rotate variant (gen_packed_body.py)

#include "generated/coupling_pk_lmax1.inc"
#include "generated/coupling_pk_lmax2.inc"
#include "generated/coupling_pk_lmax3.inc"
#include "generated/coupling_pk_lmax4.inc"
#include "generated/coupling_pk_lmax5.inc"


// ddx, ddy, ddz: components of k (r_i - r_i') (dimensionless) from the FP64 subtraction; they are rounded to FP32
// here, AFTER the subtraction (coordinate rounding is the dominant FP32 error otherwise).
// EXT (extended range): kd itself rounded to FP32 carries a phase error of kd 2^-24 rad, which reaches the 1e-4 budget
// for clusters a few thousand wavelengths across.  EXT recovers the lost part with one Newton residual in FP64,
// kd = x + (|dd|^2 - x^2) / (2 x), and hands it to the argument reduction of e^{ikd} (six FP64-pipe instructions per
// pair; everything else is unchanged).  celes_setup switches it on by the extent of the cluster.
// bload(q): emitter coefficient q in the variant's work basis;  yacc: accumulator policy of the receiver.
template <int LMAX, int VARIANT, bool TABLE, bool EXT = false, class BLoad, class YAcc>
CELES_DEVICE void pair_translate(double ddx, double ddy, double ddz, const HankelTable& htab, const BLoad& bload, YAcc& yacc) {
    constexpr int P = 2 * LMAX + 1;
    const float dx = (float)ddx, dy = (float)ddy, dz = (float)ddz;
    // ---- H2 geometry: spherical coordinates of d
    const float rho2 = fmaf(dx, dx, dy * dy);
    const float r2 = fmaf(dz, dz, rho2);
    const float rinv = rsqrtf(r2);
    const float x = r2 * rinv;                       // kd
    const float ct = dz * rinv;
    const bool on_axis = rho2 < 1e-12f * r2;         // d || z: phi := 0 (any value is right, P_p^nu(+-1) = 0 for nu > 0)
    const float rhoinv = on_axis ? 0.0f : rsqrtf(rho2);
    const float cph = on_axis ? 1.0f : dx * rhoinv;
    const float sph = on_axis ? 0.0f : dy * rhoinv;
    const float st = rho2 * rhoinv * rinv;
    // ---- H3 radial functions: h_0 = -i e^{ix}/x, h_1 = -e^{ix}(x+i)/x^2, upward recurrence (stable relative
    // to |h_p| because the Neumann part dominates wherever the Bessel part's recurrence is unstable)
    if constexpr (VARIANT == celes::kRotated && TABLE) {    // the paper's table look-up
        const float t = (x - htab.x0) * htab.inv_dx;
        const int j = min(max((int)t, 0), htab.last - 1);
        const float u = t - (float)j, v = 1.0f - u;
        const float h00 = (1.0f + 2.0f * u) * v * v, h10 = u * v * v, h01 = u * u * (3.0f - 2.0f * u), h11 = -u * u * v;
        const float4* n0 = htab.nodes + (size_t)j * P;
        float2 h[P];
#pragma unroll
        for (int p = 0; p < P; ++p) {
            const float4 a = __ldg(n0 + p), b = __ldg(n0 + P + p);
            h[p] = fma2(bc2(h11), make_float2(b.z, b.w), fma2(bc2(h01), make_float2(b.x, b.y),
                   fma2(bc2(h10), make_float2(a.z, a.w), mul2(bc2(h00), make_float2(a.x, a.y)))));
        }
        PairBodyPk<LMAX>::run(h, ct, st, cph, sph, bload, yacc);
        return;
    }
    float sx, cx, x_lo = 0.0f;
    if constexpr (EXT) {
        const double xd = (double)x;
        x_lo = (float)fma(-xd, xd, fma(ddx, ddx, fma(ddy, ddy, ddz * ddz))) * (0.5f * rinv);
    }
    sincos_kd(x, x_lo, &sx, &cx);                    // kd reaches ~1000 rad and more: reduced first
    if constexpr (VARIANT == celes::kRotated) {             // the same recurrence on packed (Re, Im)
        float2 h[P];
        h[0] = mul2(bc2(rinv), make_float2(sx, -cx));
        h[1] = fma2(bc2(rinv), h[0], nimul2(h[0]));             // h_1 = h_0 / x - e^{ix} / x,  e^{ix} / x = i h_0
#pragma unroll
        for (int p = 1; p + 1 < P; ++p) h[p + 1] = fma2(bc2((float)(2 * p + 1) * rinv), h[p], neg2(h[p - 1]));
        PairBodyPk<LMAX>::run(h, ct, st, cph, sph, bload, yacc);
    } else {
    float hr[P], hi[P];
    hr[0] = sx * rinv;
    hi[0] = -cx * rinv;
    hr[1] = fmaf(sx, rinv, -cx) * rinv;
    hi[1] = -fmaf(cx, rinv, sx) * rinv;
#pragma unroll
    for (int p = 1; p + 1 < P; ++p) {
        const float f = (float)(2 * p + 1) * rinv;
        hr[p + 1] = fmaf(f, hr[p], -hr[p - 1]);
        hi[p + 1] = fmaf(f, hi[p], -hi[p - 1]);
    }
    // ---- H4-H7 angular functions, p-contraction, n'-contraction (generated)
    PairBody<LMAX>::run(hr, hi, ct, st, cph, sph, bload, yacc);
    }
}
