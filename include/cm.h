/*
 * cm.h — C ABI of libcm: gravitational potential on nested Cartesian grids by the
 * convolution method (Vorobyov, McKevitt, Kulikov, Elbakyan, arXiv 2301.06763).
 *
 * The problem (Fig. 1; L105-L116, Eq. 9-10; L170-L186, Eq. 14):
 * `levels` concentric N^3 Cartesian grids, level 0 the coarsest (the paper's m = 1),
 * level l+1 covering the central half (coarse indices [N/4, 3N/4) per axis, L76) of
 * level l with cells of half the size, dx_l = dx0 / 2^l.  Given the density rho on
 * every level, return on every level
 *
 *     Phi(Omega^n) = Phi^{m=n} + sum_{k<n} tilde Phi_hole^{m=k}                 (Eq. 14)
 *
 * where Phi^m is the discrete sum of Eq. 10 over grid m (masses rho dx^3, inverse
 * distance between cell centres, the own-cell term of Eq. 13), Phi_hole^m the same
 * sum with the density inside the cavity set to zero (L174), both evaluated by the
 * convolution theorem on the zero-padded doubled mesh (Eq. 11), and the
 * tilde is the coarse->fine interpolation of Eq. 3-6 applied level by level.  The
 * density a coarse grid sees under a finer grid is the fine density projected onto
 * it (L280-L282).  DESIGN.md lists every reading of the paper this relies on.
 *
 * All entry points return an int status (CM_OK = 0, negative = error); none throws,
 * aborts or prints.  Pointers are DEVICE pointers unless the name says `host`.
 * There is no CPU fallback: without a CUDA device every compute call fails with
 * CM_ECUDA.
 */
#ifndef CM_H
#define CM_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct cm_plan cm_plan; /* opaque; owned by the library */

enum {
    CM_OK = 0,
    CM_EINVAL = -1,    /* bad argument (see each call) */
    CM_ENOMEM = -2,    /* device or host allocation failed */
    CM_ECUDA = -3,     /* a CUDA runtime call or kernel failed; see cm_last_cuda_error */
    CM_ENOTREADY = -4  /* cm_potential before cm_green_precompute */
};

/*
 * Create a plan for `levels` nested N^3 grids.
 *   out        : receives the plan (host pointer to a host pointer).
 *   N          : cells per axis of every level; N % 4 == 0 (the method's own requirement, L76), 16 <= N <= 512.
 *                Powers of two are the native sizes.  Any other N runs the same passes at the next power of two
 *                Nf >= N (a linear convolution needs a transform length of at least 2N - 1, L143; the surplus is more
 *                zero padding): arrays, rows, planes and the cavity geometry follow N, the spectra and K-hat follow Nf,
 *                and the cost is about that of Nf.  There are no radix-3 / radix-5 stages (the transform is radix-16
 *                in registers x radix-Nf/16 across threads), and N = 8 or 12 has no decomposition here.  Nf = 512
 *                runs the plain P3 kernel (no TMA staging, K-hat from global memory) and is not tuned like Nf <= 256.
 *   levels     : number of nested grids m >= 1 (at most 32).
 *   dx0        : cell size of level 0, > 0; dx_l = dx0 / 2^l (L48).
 *   refinement : must be 2 (the paper fixes the ratio, L42).
 * Allocates all device workspace (see cm_plan_workspace_bytes) and the twiddle
 * tables; no kernel runs.  CM_EINVAL / CM_ENOMEM / CM_ECUDA on failure, *out = NULL.
 */
int cm_plan_create(cm_plan **out, int N, int levels, double dx0, int refinement);

/*
 * Step a0 (Eq. 10, 13; L143-L147 Fig. 4): sample the dimensionless kernel
 * g(o) = 1/|o| on the rearranged doubled mesh (array index a -> offset a if a <= N,
 * else a - 2N), g(0) = 3 ln(2 + sqrt 3) - pi/2 (Eq. 13 for a cube), transform it and
 * cache the real spectrum K-hat / (2N)^3 in the plan.  One K-hat serves every level:
 * Phi^l = -G dx_l^2 (rho * g).  Idempotent; synchronises the device.
 */
int cm_green_precompute(cm_plan *plan);

/*
 * The hot path (steps a1-a8 of DESIGN.md): restriction cascade, pruned (2N)^3 FFT
 * convolution of every (level, full|hole) field with K-hat, crop, prolongation
 * cascade and the Eq. 14 sum.
 *   rho_levels : device, const, [levels][N][N][N] fp64, x fastest, level 0 coarsest,
 *                16-byte aligned.  Coarse cells under a finer grid are ignored
 *                (the projected fine density is used instead).
 *   phi_levels : device, same shape, every cell of every level overwritten.
 *                Must not alias rho_levels.
 *   stream     : a cudaStream_t (NULL = legacy default stream).  The call enqueues
 *                work and returns; no host synchronisation, no host<->device copy.
 * One solve in flight per plan.  CM_ENOTREADY before cm_green_precompute.
 */
int cm_potential(cm_plan *plan, const double *rho_levels, double *phi_levels, void *stream);

/*
 * Same computation with HOST buffers (pinned memory recommended): copies
 * rho_host -> device staging, runs cm_potential, copies the result into phi_host
 * and synchronises `stream` before returning.  Staging buffers belong to the plan
 * and are allocated on first use.  For N >= 128 the call is a level pipeline: rho is
 * copied finest level first on a plan-owned copy stream, each level's projection (a1)
 * and passes P1-P4 run under the copy of the next level, P5 + a8 run coarse -> fine at
 * the end and each level's Phi leaves for the host under the next level's P5.  Same
 * kernels, bit-identical results; for N < 128 it is copy - cm_potential - copy.
 */
int cm_potential_host(cm_plan *plan, const double *rho_host, double *phi_host, void *stream);

/*
 * The solve sharded by levels across GPUs ("each of the three steps is independent and
 * can be done in parallel"): one process per GPU, each with a plan of the WHOLE nest (same N, levels, dx0) and the
 * densities / potentials of its own contiguous levels [lo, hi) only.  A solve is three calls with two small exchanges
 * that the caller carries between neighbours (NCCL send/recv in paper_2301_06763_b200/sharded.py):
 *
 *   1. cm_shard_restrict  fine -> coarse: a1 on the own levels.  rc_from_finer (device, (N/2)^3 fp64; required iff
 *      hi < levels, else NULL) is the density of level hi projected onto the cavity of level hi-1, received from the
 *      owner of level hi; rc_to_coarser (device, (N/2)^3; iff lo > 0) receives the projection of level lo, to be sent
 *      to the owner of level lo-1.
 *   2. cm_shard_forward   P1..P4 (a2-a6) on the own levels; no exchange.
 *   3. cm_shard_finish    coarse -> fine: P5 + a8 on the own levels.  ring_from_coarser (device, (N/2+2)^3 fp64; iff
 *      lo > 0) is ext + Phi_hole of level lo-1 on its cavity grown by one cell — the box [N/4-1, 3N/4+1)^3, x fastest —
 *      received from the owner of level lo-1; ring_to_finer (device, (N/2+2)^3; iff hi < levels) receives that box of
 *      level hi-1.  phi_own is complete when the call's work on `stream` is.
 *
 *   rho_own / phi_own : device, [hi-lo][N][N][N] fp64, 16-byte aligned: levels lo .. hi-1.
 * Same kernels and the same arithmetic as cm_potential: with lo = 0, hi = levels the three calls are cm_potential, and
 * any partition gives bit-identical potentials.  The calls enqueue on `stream` and return.  CM_EINVAL for an empty or
 * out-of-range [lo, hi) or a buffer that is present when it must be NULL (or the reverse); CM_ENOTREADY before
 * cm_green_precompute.  One solve in flight per plan.
 */
int cm_shard_restrict(cm_plan *plan, const double *rho_own, int lo, int hi, const double *rc_from_finer, double *rc_to_coarser,
                      void *stream);
int cm_shard_forward(cm_plan *plan, const double *rho_own, int lo, int hi, void *stream);
int cm_shard_finish(cm_plan *plan, double *phi_own, int lo, int hi, const double *ring_from_coarser, double *ring_to_finer,
                    void *stream);

/*
 * Measurement aid: the same solve launched kernel by kernel (no graph) with CUDA
 * events recorded on `stream` between the stages; synchronises `stream` and writes
 * the stage durations in milliseconds to ms_host[0..6] (host):
 *   [0] restriction cascade (a1)   [1] P1 x forward   [2] P2 y forward
 *   [3] P3 z forward * K-hat * z inverse   [4] P4 y inverse   [5] P5 x inverse
 *   [6] prolongation + sum cascade (a8): folded into P5 (one launch per level), reported as ~0.
 * n_ms must be 7.  Results in phi_levels are identical to cm_potential's.
 */
int cm_potential_profile(cm_plan *plan, const double *rho_levels, double *phi_levels, void *stream,
                         float *ms_host, int n_ms);

/*
 * Gravitational acceleration g = -grad Phi on every level, from potentials
 * that cm_potential produced (or any potentials laid out the same way):
 *   six-point central stencil, g_x = -(Phi[i+1] - Phi[i-1]) / (2 dx_l)          (Eq. 8);
 *   method A (Eq. A.1): a neighbour outside a fine grid (level l > 0) is the ghost value
 *     interpolated from level l-1 with Eq. 3-6 (L64-L76): 3/4 Phi_c[p] + 1/4 Phi_c[p+s];
 *   method B (Eq. A.2): a neighbour that lies under the finer grid is the arithmetic
 *     mean of the potentials of its 8 children on level l+1;
 *   outer boundary of level 0 (the method has no boundary values, L164): second-order one-sided
 *     difference (paper-silent).
 *   phi_levels : device, const, [levels][N][N][N] fp64, 16-byte aligned.
 *   g_levels   : device, [levels][3][N][N][N] fp64 (component x, y, z), overwritten; must not
 *                alias phi_levels.
 * Enqueues two kernels on `stream` and returns; does not need cm_green_precompute.
 */
int cm_acceleration(cm_plan *plan, const double *phi_levels, double *g_levels, void *stream);

/*
 * The modified ("dipole") convolution method over every pair of neighbouring grids (
 * PAPER.md:L282-L288 Eq. 15, L426-L433 Eq. B.1-B.2).  The original method lets a coarse grid see the
 * finer grid's mass only through its projection, which cancels dipole moments; here, for every pair
 * n : n+1, the fine grid is expanded to the physical size of the coarse one (a doubled grid of (2N)^3
 * cells of the fine size, zero outside the fine grid), its potential is found by the same convolution
 * on a (4N)^3 padded mesh, reduced to the coarse grid (mean of the 8 fine-size cells of a coarse cell)
 * and added to the potential of the coarse grid with a cavity:
 *     Phi(Omega^n) = Phi_hole^n + reduce(Phi_dbl^{n+1}) + sum_{k<n} tilde Phi_hole^k   (n not the finest)
 *     Phi(Omega^n) = Phi^n + sum_{k<n} tilde Phi_hole^k                               (the finest grid)
 * Arguments and conventions as cm_potential.  N <= 256 (the doubled grid, 2N, must be a supported size);
 * CM_EINVAL otherwise.  The first call creates the doubled-grid plan (its K-hat: 8 (2N)^3 bytes) and
 * synchronises the device once; later calls only enqueue.  Cost: one extra (2N)^3 single-level
 * convolution per pair (the paper: x4 on CPUs, x2 with GPUs, L433).
 */
int cm_potential_modified(cm_plan *plan, const double *rho_levels, double *phi_levels, void *stream);

/*
 * The modified method with the dipole moments carried across THREE neighbouring grids (PAPER.md:L437-L448,
 * Eq. B.3-B.6, Fig. B.1):
 *     Phi(Omega^n) = Phi_hole^n + reduce(Phi_dbl,hole^{n+1}) + reduce(Phi_qdp^{n+2}) + sum_{k<n} tilde Phi_hole^k   (n < M-1)
 *     Phi(Omega^n) = Phi_hole^n + reduce(Phi_dbl^{n+1}) + sum_{k<n} tilde Phi_hole^k                              (n = M-1)
 *     Phi(Omega^n) = Phi^n + sum_{k<n} tilde Phi_hole^k                                                           (n = M)
 * The doubled grid of grid n+1 has a central hole where grid n+2 lives (its mass is not counted twice); the
 * quadrupled grid is grid n+2 expanded to the size of grid n ((4N)^3 cells of its own size), reduced by the mean over
 * the 4^3 cells of a coarse cell.  qdp_direct != 0 replaces the quadrupled grid by the direct summation of Eq. B.7
 * (cm_direct_sum; centre sampling instead of the cell mean).  N <= 128 (N <= 256 with qdp_direct), else CM_EINVAL.
 * Other arguments and conventions as cm_potential_modified.
 */
int cm_potential_modified_triplets(cm_plan *plan, const double *rho_levels, double *phi_levels, int qdp_direct, void *stream);

/*
 * Allocate what cm_potential_modified (depth = 2) or cm_potential_modified_triplets (depth = 3; qdp_direct as there)
 * needs beyond the plan itself — the single-level plans of the doubled / quadrupled grids with their K-hat, and compact
 * N^3 buffers — so that the calls themselves only enqueue (one CUDA-graph launch per call, captured on the first call per
 * (rho, phi) pair).  Optional: the two calls do the same on first use, synchronising the device once.  Idempotent;
 * all or nothing (CM_ENOMEM leaves the plan as it was).  CM_EINVAL for sizes the calls reject, CM_ENOTREADY before
 * cm_green_precompute.
 */
int cm_plan_prepare_modified(cm_plan *plan, int depth, int qdp_direct);

/*
 * Direct fine -> coarse summation (Eq. B.7): the input of grid `src_level`
 * to the potential on the coarser grid `dst_level`,
 *     Phi_ds(t) = -G sum_s rho_s dx_src^3 / |r_t - r_s|        (cell centres; all N^3 cells s of the source grid),
 * the paper's substitute for the quadrupled grid of the triplet scheme when N <= 32 (L461).  O(N^6) work.
 *   rho_levels : device, const, [levels][N][N][N]; only level src_level is read, as given (no projection).
 *   phi_dst    : device, [N][N][N] fp64, overwritten with Phi_ds on every cell of level dst_level.
 * 0 <= dst_level < src_level < levels, else CM_EINVAL.  Enqueues one kernel on `stream`.
 */
int cm_direct_sum(cm_plan *plan, const double *rho_levels, int src_level, int dst_level, double *phi_dst, void *stream);

/*
 * cm_direct_sum for callers that cannot allocate device memory (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): the same Eq. B.7 sum without a plan.  cm_direct_sum keeps its
 * per-chunk partial sums in the plan's workspace; here they live in a file-scope __device__ array of
 * CM_STATIC_SCRATCH_BYTES (4 MiB) that every GPU loading libcm holds until the process exits, so the call launches two
 * kernels and calls no cudaMalloc, cudaFree or allocating library routine.
 *   N               : cells per axis of both grids, 1 <= N <= CM_STATIC_MAX_N (the paper uses Eq. B.7 up to N = 32, L461);
 *                     larger N is rejected with CM_EINVAL and cm_static_last_error() says why.
 *   dx_src, dx_dst  : cell sizes of the source (finer) and target (coarser) grid, > 0; both grids are centred on the
 *                     origin (cell i at (i + 1/2 - N/2) dx), as nested levels are.
 *   G               : gravitational constant.
 *   rho_src         : device, const, [N][N][N] fp64, x fastest: density of the source grid, read as given.
 *   phi_dst         : device, [N][N][N] fp64, overwritten with Phi_ds on every cell of the target grid.
 *   stream          : a cudaStream_t; the call enqueues and returns.
 * The scratch array's device address is looked up once per device (cudaGetSymbolAddress, device current) — on the
 * first call, or ahead of time by cm_direct_sum_static_setup() with that device current (do that before a capture).
 * Every call on a device shares the array: it needs no clearing (a call writes every entry it later reads), but two
 * calls that overlap on the GPU (two streams, graphs replayed side by side) race on it — serialise them.
 * CM_EINVAL (size, NULL pointer, dx <= 0) or CM_ECUDA; the text is in cm_static_last_error() (thread-local, "" after
 * a call that succeeded).
 */
#define CM_STATIC_MAX_N 32
#define CM_STATIC_SCRATCH_BYTES (16u * 32u * 32u * 32u * 8u)
int cm_direct_sum_static(int N, double dx_src, double dx_dst, double G, const double *rho_src, double *phi_dst, void *stream);
int cm_direct_sum_static_setup(void);
const char *cm_static_last_error(void);

/* Release the plan and everything it owns.  NULL is accepted. */
int cm_plan_destroy(cm_plan *plan);

/* Gravitational constant used in Phi = -G sum M / r (Eq. 9-10); default 1. */
int cm_plan_set_G(cm_plan *plan, double G);

/* Device bytes owned by the plan (workspace + K-hat + tables, staging excluded). */
size_t cm_plan_workspace_bytes(const cm_plan *plan);

/* Number of kernels one cm_potential call launches (nodes of its CUDA graph). */
int cm_plan_kernel_launches(const cm_plan *plan);

/*
 * Test/diagnostic access to plan-owned intermediates of the LAST solve, copied
 * device->device into dst (device, fp64) on `stream`:
 *   CM_BUF_RESTRICTED : [levels-1][N/2]^3  projected density inside each cavity (a1)
 *   CM_BUF_HOLE       : [levels][N]^3      ext_l + Phi_hole^l (valid on the cavity
 *                                           region grown by one cell; a8's input)
 *   CM_BUF_KHAT       : [2N]^3             cached spectrum, in the library's slot order
 * n_doubles must equal the buffer's size.  CM_EINVAL otherwise.
 */
enum { CM_BUF_RESTRICTED = 0, CM_BUF_HOLE = 1, CM_BUF_KHAT = 2 };
int cm_debug_copy(cm_plan *plan, int which, double *dst, size_t n_doubles, void *stream);

/* Storage slot -> frequency index along a transformed axis of CM_BUF_KHAT (0 <= slot < 2N). */
int cm_slot_to_freq(int N, int slot);

const char *cm_error_string(int code);
/* Text of the last CUDA error seen by this plan ("" if none). */
const char *cm_last_cuda_error(const cm_plan *plan);

#ifdef __cplusplus
}
#endif
#endif /* CM_H */
