/* celes.h -- C ABI of the B200-native CELES hot path (arxiv 1706.02145, PAPER.md).
 *
 * The library solves the multiple-scattering system of N spheres, eq. (8)-(9) of the paper,
 *
 *     sum_{i',n'} M^{ii'}_{nn'} b^{i'}_{n'} = sum_{n'} T^i_{nn'} a^i_{in,n'},   M = 1 - T W,
 *
 * with the coupling operator W^{ii'}_{nn'} = A_{n'n}(r_i - r_i') (eq. 7; A from the SVWF
 * addition theorem (A.5)-(A.11)) evaluated on the fly, never stored, and the
 * sphere T-matrix diagonal T^i_{nn'} = Q^i_{tau,l} (B.1).
 *
 * Conventions
 *   - Multi-index n = (tau, l, m), tau in {1,2}, l = 1..lmax, m = -l..l; 0-based position
 *     n = (tau-1) nmax/2 + (l-1)(l+1) + (m+l), nmax = 2 lmax (lmax+2).
 *   - Coefficient vectors are complex64, interleaved (re, im), laid out [sphere i][n], length N*nmax
 *     (identical to a contiguous torch.complex64 tensor of shape [N, nmax]).
 *   - Associated Legendre functions are normalised without Condon-Shortley phase.
 *   - Lengths are in one unit U (nm in the paper's examples), k in 1/U.
 *   - Every function returns 0 (CELES_OK) or a negative error code; nothing throws, nothing is printed.
 *   - "dev" pointers are CUDA device pointers owned by the caller; "host" pointers are plain host memory.
 *     cuda_stream is a cudaStream_t (NULL = default stream).  The matvec entry points only enqueue work on
 *     that stream and do not synchronise; celes_solve and the *_host variants synchronise the stream.
 *   - There is no CPU fallback: without a CUDA device every compute entry point returns CELES_ECUDA.
 */
#ifndef CELES_H
#define CELES_H

#ifdef __cplusplus
extern "C" {
#endif

#define CELES_OK       0
#define CELES_EINVAL  -1   /* bad argument: N < 1, unsupported lmax, null pointer, non-finite input, k <= 0, overlapping spheres */
#define CELES_ENOMEM  -2   /* host or device allocation failed */
#define CELES_ECUDA   -3   /* CUDA runtime error (no device, launch failure, ...) */
#define CELES_ENOCONV -4   /* celes_solve reached max_iters; x holds the last iterate and info is filled */
#define CELES_ELIMIT  -5   /* a size beyond the fixed capacity of a no-allocation entry point (celes_far_field_noalloc) */

#define CELES_LMAX_MIN 1
#define CELES_LMAX_MAX 5   /* lmax = 5 (nmax = 70): CELES_TRANSLATION_ROTATED only */
#define CELES_MAX_HISTORY 4096

typedef struct celes_ctx celes_ctx;   /* opaque; owns every device table; freed by celes_destroy */

/* Options of celes_setup (nullable -> defaults).  Zero in a field selects its default. */
typedef struct celes_options {
    int emitter_tile;      /* emitters staged per shared-memory tile; default 32 (8 at lmax = 5) */
    int emitter_splits;    /* 0 (default): the (receiver block x emitter tile) grid is cut into runs of decreasing
                              length (see `levels`), one CTA each, dispatched in that order by the hardware;
                              S > 0: the emitter sum of every receiver block is cut into S equal slices, one CTA each.
                              Either way partial sums are added in a fixed order: results are reproducible bit for bit */
    int skip_overlap_check;/* 1: do not verify that spheres are disjoint */
    int translation;       /* how W^{ii'} b^{i'} is evaluated per pair: CELES_TRANSLATION_ROTATED (default) rotates the
                              emitter coefficients so that d is the z axis, translates along z (diagonal in m) and
                              rotates back, in packed FP32 pairs (fma.rn.f32x2);
                              CELES_TRANSLATION_DIRECT sums (A.6)-(A.8) term by term, the paper's
                              algorithm, kept as an in-library cross-check (lmax <= 4).  Same result up to FP32
                              rounding. */
    int hankel;            /* how h_p^(1)(kd) is obtained per pair: CELES_HANKEL_REGISTERS (default) evaluates e^{ikd}
                              and the upward recurrence in registers; CELES_HANKEL_TABLE is the paper's scheme
                              (PAPER.md:130): a lookup table over the radial distance with spacing hankel_dr, built by
                              celes_setup (FP64 on the host, stored FP32 on the device with the analytic derivative),
                              interpolated with cubic (Hermite) splines in the kernel.
                              Only with CELES_TRANSLATION_ROTATED. */
    double hankel_dr;      /* table spacing Delta r in the length unit U; 0 = default 1.0 (1 nm in PAPER.md:140) */
    int range;             /* FP32 validity range.  The per-pair arithmetic is FP32 after an FP64 subtraction of the
                              centres; kd rounded to FP32 carries a phase error of about kd 2^-24 rad, harmless for the
                              paper's clusters (kd < 1e3: 4e-6 relative L2 on the matvec) but equal to the 1e-4 budget
                              near kd ~ 1e4 (a cluster ~1 mm across at 550 nm).  CELES_RANGE_EXTENDED carries kd as
                              FP32 + FP64 Newton residual through the argument reduction of e^{ikd} (six more FP64
                              instructions per pair, ~1 % time), which removes that limit; CELES_RANGE_AUTO (default)
                              selects it when k x (diagonal of the centres' bounding box) exceeds
                              CELES_RANGE_AUTO_KD; CELES_RANGE_STANDARD never does.  The lookup-table mode and the
                              direct translation are standard range only. */
    int levels;            /* with emitter_splits = 0: number of levels of the guided partition.  Level 1 covers half of
                              the pair grid in SMs x CTAs/SM equal runs, level 2 a quarter, ..., the last two an equal
                              share; 1 = one wave of equal runs (fewest partial sums, ~5 % slower: of two CTAs
                              resident on an SM the warp scheduler serves one first, and the other then finishes
                              alone below full throughput); 0 = default CELES_DEFAULT_LEVELS (ten: beyond that nothing changes;
                              the halving also stops once a run would be shorter than 16 emitter tiles, which gives three
                              levels at N = 1e4 -- measured best there, the partial sums then stay in L2) */
} celes_options;
#define CELES_DEFAULT_LEVELS 10
#define CELES_RANGE_AUTO     0
#define CELES_RANGE_STANDARD 1
#define CELES_RANGE_EXTENDED 2
#define CELES_RANGE_AUTO_KD  2000.0
#define CELES_HANKEL_REGISTERS 0
#define CELES_HANKEL_TABLE     1
#define CELES_TRANSLATION_ROTATED        0
#define CELES_TRANSLATION_DIRECT         1

#define CELES_GMRES    0
#define CELES_BICGSTAB 1
#define CELES_PRECOND_NONE      0
#define CELES_PRECOND_BLOCKDIAG 1
typedef struct celes_solve_opts {
    int method;            /* CELES_GMRES or CELES_BICGSTAB, the paper's two solvers */
    int restart;           /* GMRES restart length; default 30 */
    double rtol;           /* stop when ||T a_in - M x||_2 / ||T a_in||_2 <= rtol; default 1e-4 */
    int max_iters;         /* bound on inner iterations (= system matvecs inside cycles); default 1000 */
    int precond;           /* CELES_PRECOND_NONE (default) or CELES_PRECOND_BLOCKDIAG: right preconditioning with the
                              block-diagonal operator of celes_precond_setup; the stopping
                              criterion stays the TRUE residual of the unpreconditioned system */
} celes_solve_opts;

typedef struct celes_precond_info {
    int n_groups;             /* number of non-empty cuboids N_G */
    int max_group_spheres;    /* largest N_j */
    long long block_bytes;    /* device memory of the stored blocks, 8 * sum_j (N_j nmax)^2 */
    double seconds;           /* wall-clock time of celes_precond_setup */
} celes_precond_info;

typedef struct celes_solve_info {
    int iterations;        /* inner GMRES iterations / BiCGSTAB iterations (two system matvecs each) performed */
    int matvecs;           /* system matvecs, including the true-residual evaluations at restarts */
    int converged;         /* 1 if the TRUE relative residual met rtol */
    double rel_residual;   /* true relative residual ||T a_in - M x|| / ||T a_in|| of the returned x */
    double seconds;        /* wall-clock time inside celes_solve */
    int n_history;         /* entries used in history */
    double history[CELES_MAX_HISTORY]; /* relative residual estimate after each inner iteration */
} celes_solve_info;

/* celes_setup -- particle positions, radii, Mie coefficients, k and lmax.
 *   pos_xyz  host, [N][3] double, sphere centres r_i.
 *   radii    host, [N] double, R_i; used only to verify that spheres are disjoint (needed for |r| < |d| in A.5).
 *   mie_q    host, [N][2][lmax] complex128 interleaved: Q^i_{tau,l} of (B.2)-(B.3).
 *   k        background wavenumber n_0 omega / c > 0.
 * Builds on the device: k-scaled FP64 centres, the T diagonal and, if asked for, the spherical-Hankel lookup table
 * (PAPER.md:130); the a5/b5 translation coefficients are immediates of the generated pair
 * bodies and a device table for the preconditioner's block assembly.  Copies everything it needs; the host arrays
 * may be freed afterwards.
 * On success *out is a new context; on error *out is NULL. */
int celes_setup(celes_ctx** out, int N, int lmax, const double* pos_xyz, const double* radii,
                const double* mie_q, double k, const celes_options* opt, void* cuda_stream);

/* y = W b : y^i_n = sum_{i' != i} sum_{n'} W^{ii'}_{nn'} b^{i'}_{n'}  (eq. 6 without a_in).
 * b_dev, y_dev: device, N*nmax complex64, must not alias.  Asynchronous on cuda_stream. */
int celes_coupling_matvec(celes_ctx* ctx, const void* b_dev, void* y_dev, void* cuda_stream);

/* out = M b = b - T (W b)  (eqs. 8-9).  Same argument rules as above. */
int celes_system_matvec(celes_ctx* ctx, const void* b_dev, void* out_dev, void* cuda_stream);

/* Receiver-row slices of the two products: rows [row_begin, row_end) of y = W b (or of b - T (W b)) from the FULL
 * vector b -- the compute half of a receiver-sharded deployment, where every rank owns a slice of the rows and needs
 * every emitter's coefficients (the paper itself is single-GPU).
 *   b_dev        device, N*nmax complex64, all spheres.
 *   y_rows_dev   device, (row_end - row_begin)*nmax complex64: rows row_begin.. of the result.
 * The work partition and the order of the partial sums are those of the full product restricted to the receiver
 * blocks that hold the rows, so slices concatenate to the full result bit for bit.  0 <= row_begin < row_end <= N.
 * Asynchronous on cuda_stream. */
int celes_coupling_matvec_rows(celes_ctx* ctx, int row_begin, int row_end, const void* b_dev, void* y_rows_dev,
                               void* cuda_stream);
int celes_system_matvec_rows(celes_ctx* ctx, int row_begin, int row_end, const void* b_dev, void* out_rows_dev,
                             void* cuda_stream);

/* Host-buffer variants: copy b from host memory (pinned or pageable), run the device path, copy the result back,
 * synchronise.  b_host, y_host: N*nmax complex64. */
int celes_coupling_matvec_host(celes_ctx* ctx, const void* b_host, void* y_host, void* cuda_stream);
int celes_system_matvec_host(celes_ctx* ctx, const void* b_host, void* out_host, void* cuda_stream);

/* Solve eq. (8) for the scattered-field coefficients b with a host-driven Krylov loop whose matvecs, dot products,
 * axpys and norms are device kernels.
 *   a_in_dev  device, N*nmax complex64: initial-field coefficients a_in (the library forms T a_in).
 *   x_dev     device, N*nmax complex64: in = initial guess x0 (zero it for x0 = 0), out = b.
 *   o         nullable -> defaults (GMRES(30), rtol 1e-4, 1000 iterations).
 *   info      nullable.
 * Returns CELES_OK, or CELES_ENOCONV with x and info still filled. */
int celes_solve(celes_ctx* ctx, const void* a_in_dev, void* x_dev, const celes_solve_opts* o,
                celes_solve_info* info, void* cuda_stream);

/* Block-diagonal preconditioner (Fig. 1).  The spheres are divided into subsets G_j by an array
 * of cuboids with edge lengths edge_xyz[3] (unit U; an edge <= 0 means "do not cut along that axis") anchored at the
 * minimum corner of the centres' bounding box; for every subset the dense block M_j = (1 - T W) restricted to G_j
 * is assembled on the device and eliminated with partial (row) pivoting through to its inverse (a blocked Gauss-Jordan
 * elimination in the library's own kernels, all blocks side by side); the context stores the inverses
 * (8 * sum_j (N_j nmax)^2 bytes; the elimination runs in place).  Replaces an earlier preconditioner of
 * the context, reusing its device memory if the new one fits (no allocator call then).  Synchronises the device.
 * CELES_EINVAL: bad argument or a subset with more than 25600 / nmax spheres; CELES_ENOMEM: blocks do not fit;
 * CELES_ECUDA: CUDA failure or a singular block. */
int celes_precond_setup(celes_ctx* ctx, const double* edge_xyz, celes_precond_info* info, void* cuda_stream);

/* z = blockdiag(M_j^{-1}) v (step 4 of PAPER.md:114).  v_dev, z_dev: device, N*nmax complex64, must not alias.
 * Asynchronous on cuda_stream.  CELES_EINVAL if celes_precond_setup has not succeeded on this context. */
int celes_precond_apply(celes_ctx* ctx, const void* v_dev, void* z_dev, void* cuda_stream);

/* Host-only (needs no GPU): the cuboid partition celes_precond_setup uses.  pos_xyz host [N][3], edge_xyz host [3];
 * group_of[i] (host, [N]) receives the subset of sphere i, subsets numbered in lexicographic (cx, cy, cz) order of
 * the non-empty cuboids; *n_groups (nullable) their number. */
int celes_partition(int N, const double* pos_xyz, const double* edge_xyz, int* group_of, int* n_groups);

/* Far field of the scattered field (PAPER.md:271 (A.12), 351-369 (D.1)-(D.3)): every sphere's outgoing SVWFs are turned
 * into plane waves about its own centre with (A.12) and the contributions are added:
 *     g_j(alpha, beta) = (1 / 2 pi) sum_i exp(-i k(alpha,beta).r_i) sum_n b^i_n B_nj(beta) exp(i m alpha),  j = 1, 2,
 * with B_nj of (A.14) and k(alpha,beta) = k (sin beta cos alpha, sin beta sin alpha, cos beta); the radiant intensity is
 * I_j = 2 pi^2 / (omega k mu_0) |g_j|^2 (D.3).
 *   b_dev   device, N*nmax complex64: scattered-field coefficients (e.g. the solution of celes_solve).
 *   alpha, beta  host, [n_dir] double: azimuthal and (real) polar angles of the directions, radians.
 *   g_dev   device, [n_dir][2] complex64: g_1, g_2 per direction.
 * Asynchronous on cuda_stream: the direction tables live in a scratch block that the context keeps and reuses (a call
 * that needs a larger block than any before it synchronises the stream once to grow it).  alpha and beta are read
 * before the call returns if they are pageable memory; pinned arrays must stay valid until the stream has run.
 * The field calls of one context share that scratch block: issue them on one stream. */
int celes_far_field(celes_ctx* ctx, const void* b_dev, int n_dir, const double* alpha, const double* beta,
                    void* g_dev, void* cuda_stream);

/* celes_far_field for callers that must not allocate (code under CUDA graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc): same arguments, same result, but every table the kernels need (directions, B_nj e^{i m alpha}, the
 * split partial sums of the sphere sum) lives in ONE static device array of the library -- 5 MiB, held by every GPU that
 * loads the library until the process exits -- whose device address celes_setup looked up once for the context's device.
 * The call makes no cudaMalloc, no cudaFree and no host allocation, whatever it was called with before.
 *   n_dir <= CELES_FAR_FIELD_NOALLOC_MAX_DIR (2048), any supported lmax; more directions: CELES_ELIMIT, nothing is launched
 *   (evaluate them in batches, or use celes_far_field).
 * The array is shared by every context and every call on the device and keeps the previous call's contents; nothing in it
 * has to start at zero (each call overwrites every entry it reads).  Two calls that overlap on the GPU (different streams,
 * or different host threads on one device) RACE on it: issue them on one stream, or order them with events.
 * alpha, beta: host arrays, copied with cudaMemcpyAsync on cuda_stream (pinned memory keeps the call asynchronous).
 * Errors as celes_far_field, plus CELES_ELIMIT; CELES_ECUDA if the array's address could not be resolved at set-up. */
#define CELES_FAR_FIELD_NOALLOC_MAX_DIR 2048
int celes_far_field_noalloc(celes_ctx* ctx, const void* b_dev, int n_dir, const double* alpha, const double* beta,
                            void* g_dev, void* cuda_stream);

/* Initial-field coefficients of the plane wave E_0 Phi_j(alpha, beta; r) = E_0 exp(i k.r) e_j about every sphere centre,
 * from (A.13)-(A.14): a^i_n = E_0 exp(i k.r_i) 4 exp(-i m alpha) B^dagger_nj(beta).
 *   alpha, beta   azimuthal and polar angle of the wave vector, radians (beta = 0: propagation along +z).
 *   polarisation  j = 1: along e_alpha (TE), j = 2: along e_beta (TM; x-polarised for alpha = beta = 0).
 *   a_in_dev      device, N*nmax complex64.  Asynchronous on cuda_stream. */
int celes_plane_wave(celes_ctx* ctx, double alpha, double beta, int polarisation, double E0_re, double E0_im,
                     void* a_in_dev, void* cuda_stream);

/* Gaussian beam of Appendix C: waist w centred at r_G, propagating along +z, field at the waist
 * E_0 (-sin alpha_G e_x + cos alpha_G e_y) exp(-((x-x_G)^2 + (y-y_G)^2)/w^2) (C.1). */
typedef struct celes_beam {
    double waist;          /* w > 0, length unit U */
    double center[3];      /* r_G */
    double alpha_G;        /* polarisation angle, radians */
    double E0_re, E0_im;   /* complex amplitude E_0 */
    int n_beta;            /* Gauss-Legendre nodes of the polar-angle integral over [0, pi/2]; 0 = default 400 */
} celes_beam;

/* Initial-field coefficients a_in of the beam about every sphere centre, (C.8) with the analytic azimuthal integral
 * (C.7), evaluated on the device in FP64 and rounded once.  a_in_dev: device, N*nmax complex64 (the
 * input of celes_solve).  Asynchronous on cuda_stream (scratch block of the context, see celes_far_field). */
int celes_gaussian_beam(celes_ctx* ctx, const celes_beam* beam, void* a_in_dev, void* cuda_stream);

/* Scattered electric field at n_pts points, eq. (3) with the explicit outgoing SVWFs (A.2):
 *     E_scat(r) = sum_i sum_n b^i_n Psi^(3)_n(r - r_i)          (the near-field maps of Figs. 2 and 6).
 *   b_dev    device, N*nmax complex64.
 *   pts_xyz  host, [n_pts][3] double, unit U.  The expansion of sphere i holds for |r - r_i| > R_i only: points inside
 *            a sphere get the (meaningless) analytic continuation, not the internal field.
 *   e_dev    device, [n_pts][3] complex64: Cartesian components (x, y, z).
 * Asynchronous on cuda_stream (scratch block of the context, see celes_far_field). */
int celes_scattered_field(celes_ctx* ctx, const void* b_dev, int n_pts, const double* pts_xyz, void* e_dev,
                          void* cuda_stream);

/* Release the context and every device table it owns.  NULL is allowed. */
void celes_destroy(celes_ctx* ctx);

/* Static description of an error code. */
const char* celes_strerror(int code);

/* Sizes the caller needs: nmax = 2 lmax (lmax+2); returns CELES_EINVAL (<0) for an unsupported lmax. */
int celes_nmax(int lmax);

/* Launch geometry of the coupling kernel of this context (for reporting): receiver blocks, the caller's fixed
 * emitter splits (0 = guided partition), threads per block, emitters per tile.  Any pointer may be NULL. */
int celes_launch_config(const celes_ctx* ctx, int* receiver_blocks, int* emitter_splits, int* block_threads,
                        int* emitter_tile);

/* Numerical range of this context (for reporting): kd_max = k x diagonal of the centres' bounding box, and whether the
 * extended range mode of celes_options.range is active (1) or not (0).  Any pointer may be NULL. */
int celes_range_info(const celes_ctx* ctx, double* kd_max, int* extended);

/* Work partition of the coupling kernel (for reporting): CTAs launched for a full product, segments (= partial-sum
 * slots of N_block x nmax complex64 each) and receivers per receiver block.  Any pointer may be NULL. */
int celes_work_partition(const celes_ctx* ctx, int* ctas, int* segments, int* receivers_per_block);

/* Host-only (needs no GPU): the work partition celes_setup builds for N spheres, emitter tiles of emitter_tile,
 * resident_ctas = SMs x CTAs/SM, and levels / emitter_splits as in celes_options.  seg_out (nullable, host,
 * [seg_capacity][5] int) receives one row (cta, receiver block, e_begin, e_end, slot) per segment in launch order. */
int celes_plan_work(int N, int emitter_tile, int resident_ctas, int levels, int emitter_splits, int* ctas, int* segments,
                    int* receivers_per_block, int* seg_out, int seg_capacity);

/* Host-only (needs no GPU): the translation coefficients the library uses, for W_{(tau l m),(tau' l' m')}:
 *   a5_re[((r*H)+c)*P + p] = Re a5(l',m'|l,m|p),  b5_im[...] = Im b5(l',m'|l,m|p)   (eq. 7),
 * r, c = (l-1)(l+1)+(m+l) of receiver / emitter, H = lmax (lmax+2), P = 2 lmax + 1, p = 0..2 lmax.
 * Both arrays have H*H*P doubles. */
int celes_translation_table(int lmax, double* a5_re, double* b5_im);

#ifdef __cplusplus
}
#endif
#endif /* CELES_H */
