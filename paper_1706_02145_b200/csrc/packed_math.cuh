// packed_math.cuh -- small device helpers shared by every kernel file: packed FP32 pairs and the reduced sine / cosine.
#pragma once
#include <cuda_runtime.h>

#ifndef CELES_DEVICE
#define CELES_DEVICE __device__ __forceinline__
#endif

// Packed FP32 pairs (sm_100a: fma.rn.f32x2 / mul.rn.f32x2 / add.rn.f32x2 -> SASS FFMA2 / FMUL2 / FADD2).  A float2
// holds one complex number (re, im); bc2(a) is the broadcast operand (a, a), which ptxas encodes as a scalar
// register operand of FFMA2, and negations / swapped halves fold into operand modifiers.
CELES_DEVICE float2 bc2(float a) { return make_float2(a, a); }
CELES_DEVICE float2 neg2(float2 a) { return make_float2(-a.x, -a.y); }
CELES_DEVICE float2 fma2(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }
CELES_DEVICE float2 mul2(float2 a, float2 b) { return __fmul2_rn(a, b); }
CELES_DEVICE float2 add2(float2 a, float2 b) { return __fadd2_rn(a, b); }
CELES_DEVICE float2 sub2(float2 a, float2 b) { return __fadd2_rn(a, neg2(b)); }
// i a and -i a: swapped halves with a (-,+) / (+,-) sign pattern, which FFMA2 / FADD2 take as operand modifiers
// (SASS .LO_HI / .NP) on their vector operands -- no instruction of their own.
CELES_DEVICE float2 imul2(float2 a) { return make_float2(-a.y, a.x); }
CELES_DEVICE float2 nimul2(float2 a) { return make_float2(a.y, -a.x); }
// Complex multiply(-add) k x (+ c) in TWO packed instructions: the broadcast scalar operand cannot carry the
// (-k.y, +k.y) pattern, but the addend can be read as (-c.x, c.y) and the vector multiplicand with swapped halves:
//   t = k.y (x.y, x.x) + (-c.x, c.y) = (-Re, Im) of c + i k.y x;   k.x x + (-t.x, t.y) = c + k x.
CELES_DEVICE float2 cfma2(float2 k, float2 x, float2 c) {
    const float2 t = __ffma2_rn(bc2(k.y), make_float2(x.y, x.x), make_float2(-c.x, c.y));
    return __ffma2_rn(bc2(k.x), x, make_float2(-t.x, t.y));
}
CELES_DEVICE float2 cmul2(float2 k, float2 x) {
    const float2 t = __fmul2_rn(bc2(k.y), make_float2(x.y, x.x));
    return __ffma2_rn(bc2(k.x), x, make_float2(-t.x, t.y));
}

// sin, cos of kd.  kd reaches ~1e3 rad, where the hardware approximations (MUFU.SIN / MUFU.COS behind __sincosf) are
// useless on their own; after a Cody-Waite reduction to [-pi, pi] (2 pi = 6.28125 + 1.9353072e-3: the first product
// n * 6.28125 is exact for n < 2^15) their absolute error is ~4e-7, far inside the 1e-4 budget, and the pair saves the
// ~25 instructions of sincosf's polynomial path.  Define CELES_ACCURATE_SINCOS to get sincosf back.
// x_lo: the part of kd that FP32 x does not hold (0 in the standard range mode); it is added AFTER the reduction,
// where it is not absorbed by the rounding of x.
CELES_DEVICE void sincos_kd(float x, float x_lo, float* s, float* c) {
#ifdef CELES_ACCURATE_SINCOS
    sincosf(x + x_lo, s, c);
#else
    const float n = rintf(x * 0.15915494309189535f);
    float r = fmaf(n, -6.28125f, x);
    r = fmaf(n, -1.9353071795864769e-3f, r) + x_lo;
    __sincosf(r, s, c);
#endif
}
