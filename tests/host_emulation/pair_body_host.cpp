// Host emulation of the generated pair bodies (tests only): compiles csrc/pair_math.cuh and the generated
// coupling_*_lmax*.inc with g++ by defining the handful of device intrinsics they use, so that the straight-line code
// the generators write can be checked against the FP64 oracle on a machine without a GPU (tests/test_host_logic.py).
// Same FP32 operation order as the device code (fmaf for every FMA); rsqrt and sin / cos are the libm ones.
#include <cmath>
#include <cuda_runtime.h>   // float2 / float4, make_float2 (host definitions)

#define CELES_DEVICE inline
static inline float2 __ffma2_rn(float2 a, float2 b, float2 c) { return make_float2(fmaf(a.x, b.x, c.x), fmaf(a.y, b.y, c.y)); }
static inline float2 __fmul2_rn(float2 a, float2 b) { return make_float2(a.x * b.x, a.y * b.y); }
static inline float2 __fadd2_rn(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
static inline float celes_host_rsqrtf(float x) { return 1.0f / sqrtf(x); }
static inline void celes_host_sincosf(float x, float* s, float* c) { *s = sinf(x); *c = cosf(x); }
static inline float4 celes_host_ldg(const float4* p) { return *p; }
#define rsqrtf celes_host_rsqrtf
#define __sincosf celes_host_sincosf
#define __ldg celes_host_ldg
using std::min;
using std::max;

#include "pair_math.cuh"

namespace {
template <int NMAX>
struct YHost {
    float2 y[NMAX];
    void operator()(int q, float r, float i) { y[q].x += r; y[q].y += i; }
    float2 get(int q) const { return y[q]; }
    void put(int q, float2 v) { y[q] = v; }
};

template <int LMAX, int VARIANT>
void run(float dx, float dy, float dz, const float2* b, float2* y) {
    constexpr int NMAX = 2 * LMAX * (LMAX + 2);
    YHost<NMAX> acc;
    for (int q = 0; q < NMAX; ++q) acc.y[q] = y[q];
    HankelTable none = {nullptr, 0.0f, 0.0f, 0};
    auto bload = [b](int q) { return b[q]; };
    pair_translate<LMAX, VARIANT, false>(dx, dy, dz, none, bload, acc);
    for (int q = 0; q < NMAX; ++q) y[q] = acc.y[q];
}
}  // namespace

// y[nmax] += W_work(k d) b[nmax]: one pair, both vectors in the variant's WORK basis (pack_kernel's output layout),
// complex64 interleaved.  variant: 0 packed rotated, 1 direct.  Returns 0, or -1 for an unsupported (lmax, variant).
extern "C" int celes_host_pair_body(int lmax, int variant, float kdx, float kdy, float kdz, const float* b, float* y) {
    const float2* bb = reinterpret_cast<const float2*>(b);
    float2* yy = reinterpret_cast<float2*>(y);
    switch (lmax * 2 + variant) {
        case 2: run<1, 0>(kdx, kdy, kdz, bb, yy); return 0;
        case 3: run<1, 1>(kdx, kdy, kdz, bb, yy); return 0;
        case 4: run<2, 0>(kdx, kdy, kdz, bb, yy); return 0;
        case 5: run<2, 1>(kdx, kdy, kdz, bb, yy); return 0;
        case 6: run<3, 0>(kdx, kdy, kdz, bb, yy); return 0;
        case 7: run<3, 1>(kdx, kdy, kdz, bb, yy); return 0;
        case 8: run<4, 0>(kdx, kdy, kdz, bb, yy); return 0;
        case 9: run<4, 1>(kdx, kdy, kdz, bb, yy); return 0;
        case 10: run<5, 0>(kdx, kdy, kdz, bb, yy); return 0;
    }
    return -1;
}
