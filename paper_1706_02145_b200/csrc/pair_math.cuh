// pair_math.cuh -- per-pair arithmetic of the direct coupling kernel (steps H2-H7 of DESIGN.md).
//
// For the ordered pair (receiver i, emitter i') with d = r_i - r_i' (eq. 7) this evaluates
// h_p^(1)(kd), P_p^nu(cos theta_d), e^{i nu phi_d} in registers and applies the 2x2 tau-block translation
// (A.6)-(A.8), to the emitter's coefficients.  The contraction itself is generated code
// (generated/coupling_body_lmax*.inc, written by gen_coupling_body.py).
#pragma once

#ifndef CELES_DEVICE
#define CELES_DEVICE __device__ __forceinline__
#endif

template <int LMAX>
struct PairBody;   // specialised by the generated files

#include "generated/coupling_body_lmax1.inc"
#include "generated/coupling_body_lmax2.inc"
#include "generated/coupling_body_lmax3.inc"
#include "generated/coupling_body_lmax4.inc"

template <int LMAX>
struct PairBodyRot;   // rotate / axial-translate / rotate variant (gen_rotated_body.py)

#include "generated/coupling_rot_lmax1.inc"
#include "generated/coupling_rot_lmax2.inc"
#include "generated/coupling_rot_lmax3.inc"
#include "generated/coupling_rot_lmax4.inc"

// dx, dy, dz: components of k (r_i - r_i') (dimensionless), already rounded to FP32 AFTER the subtraction
// was done in FP64 (coordinate rounding is the dominant FP32 error otherwise).
// bload(q): emitter coefficient q of [b_+ | b_-];  yacc(q, re, im): y_pm[q] += (re, im).
template <int LMAX, bool ROTATED, class BLoad, class YAcc>
CELES_DEVICE void pair_translate(float dx, float dy, float dz, const BLoad& bload, YAcc& yacc) {
    constexpr int P = 2 * LMAX + 1;
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
    float sx, cx;
    sincosf(x, &sx, &cx);                            // full-range accurate: kd reaches ~1000 rad
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
    if (ROTATED) PairBodyRot<LMAX>::run(hr, hi, ct, st, cph, sph, bload, yacc);
    else PairBody<LMAX>::run(hr, hi, ct, st, cph, sph, bload, yacc);
}
