// ctx.h -- the context behind the opaque celes_ctx* of include/celes.h, and the few internal host functions that
// the translation units of the library share (celes.cu: set-up and matvec; solve.cu: GMRES / BiCGSTAB; precond.cu:
// block-diagonal preconditioner; fields.cu: Gaussian beam, far field, near field).
#pragma once
#include <cuda_runtime.h>

#include <new>
#include <vector>

#include "../../include/celes.h"
#include "hankel_table.h"
#include "variants.h"

struct celes_ctx {
    int N = 0, lmax = 0, nmax = 0;
    double k = 0.0;
    int device = 0, sm_count = 0;
    int etile = 32;
    // work partition of the coupling kernel (work_partition.h): receiver blocks of bs spheres, n_cta CTAs walking
    // n_seg segments, one partial-sum slot per segment
    int bs = 0, rblocks = 0, n_cta = 0, n_seg = 0, fixed_splits = 0;
    int* cta_begin = nullptr;    // [n_cta + 1]
    int4* seg = nullptr;         // [n_seg] (rblock, e_begin, e_end, slot)
    int* slot_begin = nullptr;   // [rblocks + 1]
    std::vector<int> h_cta_of_block_first, h_cta_of_block_last;   // [rblocks] first / last CTA with a segment of the block
    bool extended_range = false; // kd carried as FP32 + residual (pair_math.cuh, EXT); chosen by celes_setup
    double kd_max = 0.0;         // k x diagonal of the centres' bounding box
    int variant = celes::kRotated;   // CELES_TRANSLATION_*: packed rotated (default), direct sum, scalar rotated
    size_t coupling_smem = 0;
    std::vector<double> pos;     // host copy of the centres [N][3] (partition of the preconditioner)
    double* kpos = nullptr;      // [N][3] FP64, k * r_i
    float2* tdiag = nullptr;     // [N][nmax] T diagonal Q^i_{tau,l} expanded over m (B.1)
    float4* htab = nullptr;      // Hankel lookup table [nodes][2 lmax + 1] (CELES_HANKEL_TABLE), else null
    HankelTable htab_desc = {nullptr, 0.0f, 0.0f, 0};
    float2* bpm = nullptr;       // [N][nmax] work: [b_+ | b_-]
    float2* ypart = nullptr;     // [n_seg][kBlock][nmax] work: partial sums, one slot per segment
    void* far_static = nullptr;  // device address of the static scratch of celes_far_field_noalloc on this context's device
    void* scratch = nullptr;     // device scratch of the field calls (direction / beam / point tables), grown on demand
    size_t scratch_bytes = 0;
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
    long long pc_capacity = 0;   // elements allocated behind pc_blocks (a later set-up that fits reuses the buffer)
    char* pc_arena = nullptr;    // one allocation behind every index / work array of the preconditioner (and the set-up's
    size_t pc_arena_bytes = 0;   // temporaries): grow-only, so a set-up that replaces an earlier one calls no allocator
    int* pc_order = nullptr;     // [N]
    int* pc_grp_offset = nullptr;        // [groups+1]
    long long* pc_blk_offset = nullptr;  // [groups]
    int* pc_cta_group = nullptr;         // [pc_ctas]
    int* pc_cta_row0 = nullptr;          // [pc_ctas]
    int* pc_perm = nullptr;              // [N nmax] row permutation P_j of every block's pivoted elimination
    float2* pc_blocks = nullptr;         // B_j = M_j^{-1} P_j^T, column-major, back to back
    float2* pc_tmp = nullptr;            // [n] work vector of the preconditioned solve
};

#define CU_TRY(expr)                                  \
    do {                                              \
        cudaError_t e_ = (expr);                      \
        if (e_ != cudaSuccess) {                      \
            return e_ == cudaErrorMemoryAllocation ? CELES_ENOMEM : CELES_ECUDA; \
        }                                             \
    } while (0)

// Nothing may throw across the C ABI (celes.h): every extern "C" body that allocates host memory runs inside this.
#define CELES_NOTHROW(call)                                  \
    try { return (call); }                                   \
    catch (const std::bad_alloc&) { return CELES_ENOMEM; }   \
    catch (...) { return CELES_ECUDA; }

namespace celes {
namespace host {
// rows [row_begin, row_end) of y = W b (system == false) or out = b - T (W b): pack -> coupling -> finalize, all on
// stream s; b is the full vector, out holds the rows only (celes.cu)
int run_matvec(celes_ctx* c, const float2* b, float2* out, bool system, cudaStream_t s, int row_begin, int row_end);
inline int run_matvec(celes_ctx* c, const float2* b, float2* out, bool system, cudaStream_t s) {
    return run_matvec(c, b, out, system, s, 0, c->N);
}
// z = blockdiag(M_j^{-1}) v, and release of the preconditioner (precond.cu)
int precond_apply(celes_ctx* c, const float2* v, float2* z, cudaStream_t s);
void free_precond(celes_ctx* c);
// device address of fields.cu's static scratch array on the current device, one cudaGetSymbolAddress per device (fields.cu)
int far_static_scratch_address(int device, void** out);
// release of the Krylov work space (solve.cu)
void free_krylov(celes_ctx* c);
}  // namespace host
}  // namespace celes
