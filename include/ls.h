/* ls.h — C ABI of libls.so: the narrow-band level-set hot path on one B200 (sm_100a).
 *
 * Method: arxiv/paper_1612_04040 ("Parallel Level set algorithm with MPI and accelerated on GPU").
 * Citations are /root/reference/PAPER.md line numbers plus the equation / step they fall in;
 * "R<n>" are the readings listed in DESIGN.md (where the paper is silent or garbled).
 *
 * Conventions that hold for every call
 *   - Fields are dense 3-D arrays, x fastest: idx = (k*ny + j)*nx + i       (§3).
 *     Element type is the ctx dtype (float or double), nx*ny*nz elements.
 *   - `phi`, `F`, `out`, `d`, `phi_bar` are DEVICE pointers owned by the caller, aligned to at
 *     least 16 bytes (any cudaMalloc / torch allocation is), alive until the ctx stream drained.
 *     Only ls_step_host, ls_band_counts, ls_band_export, ls_stats and the out-parameters of
 *     ls_reinit_tol take HOST pointers; each says so.
 *   - All work is enqueued on the stream given to ls_create; calls return without waiting unless
 *     stated ("synchronises").  One ctx <-> one stream; a ctx is not thread-safe.
 *   - Scalars arrive as double and are rounded ONCE to the field type; all per-point arithmetic is
 *     in the field type with IEEE divide / square root and no FMA contraction (R18).
 *   - Domain boundary: edge replicate — a neighbour index outside [0, n-1] is clamped (R3).
 *   - 8x8x8 bricks: NB* = ceil(n* / 8), brick id b = (bz*NBy + by)*NBx + bx; per brick 8 uint64
 *     mask words, word lz (0..7), bit ly*8 + lx; cells outside the domain have bit 0 (R20).
 *   - Every call returns an ls_status; nothing aborts or throws.  CUDA faults that surface
 *     asynchronously are reported as LS_ERR_CUDA by the next call that synchronises.
 *   - Preconditions NOT checked: finite inputs; max|F|*dt < dx ("the front moves less than one
 *     grid point").
 *   - There is no CPU fallback anywhere: with no usable CUDA device every call that needs one
 *     returns LS_ERR_CUDA.
 */
#ifndef LS_H_
#define LS_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    LS_OK = 0,
    LS_ERR_ARG = 1,       /* null pointer, non-positive dx, negative iters, beta >= gamma (finite), ... */
    LS_ERR_DIM = 2,       /* a grid dimension < 1, or the grid too large for int32 brick ids */
    LS_ERR_DTYPE = 3,     /* dtype not LS_F32 / LS_F64 */
    LS_ERR_ALLOC = 4,     /* device or host allocation failed */
    LS_ERR_CUDA = 5,      /* a CUDA runtime call failed (ls_last_cuda_error has the text) */
    LS_ERR_CAPACITY = 6,  /* internal list capacity exceeded (cannot happen: lists are sized for all bricks) */
    LS_NOT_CONVERGED = 7, /* ls_reinit_tol reached max_iters; the result is still valid */
    LS_ERR_STATE = 8      /* a band call before any ls_build_band */
} ls_status;

typedef enum { LS_F32 = 0, LS_F64 = 1 } ls_dtype;

/* How ls_step performs Step 1 on the 2nd and later steps of one call. */
typedef enum {
    LS_REBUILD_FULL = 0,        /* scan every grid point each step, as the paper does */
    LS_REBUILD_INCREMENTAL = 1  /* exact: after the first step phi is clamped (eq. 10), so
                                   T^{n+1} is a subset of N^n and only the bricks of N^n
                                   are re-classified — fused into the launch that writes phi^{n+1}: the
                                   last reinit sweep, or (iters even or 0) the band copy that moves the
                                   result; either way no whole-grid pass after the first step */
} ls_rebuild;

/* Parameters of one narrow-band step (Steps 1-3). */
typedef struct {
    double dx;    /* grid spacing, > 0 */
    double dt;    /* time step of eq. 3/8 */
    double dtau;  /* pseudo-time step of eq. 12 */
    double beta;  /* cut-off: c = 1 for |phi| <= beta            (eq. 7) */
    double gamma; /* tube half-width: T = {|phi| < gamma}         (eq. 6); 0 < beta < gamma */
    int32_t iters;   /* reinitialisation iterations per step, >= 0 (R13) */
    int32_t rebuild; /* ls_rebuild */
    int32_t chained; /* 0 or 1.  1 = the caller promises that `phi` is the same buffer, unmodified, that
                        the previous ls_step on this ctx returned (same gamma), and that no other band
                        call was made on the ctx in between.  The ctx then keeps its band, its scratch
                        field and (LS_REBUILD_INCREMENTAL) the T masks it emitted from phi^n, so the call
                        does no whole-grid work at all: no resync copy, no scan, no global clamp.  If the
                        ctx cannot verify pointer / gamma / state it silently runs the unchained path. */
    int32_t fuse;     /* reinit sweeps per kernel launch: 0 = library default (1), 1 = one launch per sweep, 2 = two
                         sweeps per launch where the grid allows it (temporal blocking of eq. 12's iterations in
                         shared memory: the tile is loaded once, sweep k is evaluated on the tile's N points and on
                         the one-cell ring around it, sweep k+1 on the tile's own points).  The results do not
                         depend on it: Jacobi order is kept exactly.  One sweep per launch is the default because it
                         is the faster one on B200 (the sweeps are bound by instruction issue, not by memory traffic,
                         and the ring costs extra evaluations: DESIGN.md section 6). */
} ls_params;

/* Kernel classes of the per-kernel device timing (ls_profile_*). */
typedef enum {
    LS_K_CLASSIFY = 0, /* whole-grid |phi| < gamma sweep of Step 1 */
    LS_K_BAND = 1,     /* dilation + ordered compaction of the brick lists */
    LS_K_ADVANCE = 2,  /* Step 2 */
    LS_K_REINIT = 3,   /* one Step 3 sweep (clamp / T emission fused into the last) */
    LS_K_CLAMP = 4,    /* eq. 10 passes outside the reinit sweeps */
    LS_K_COPY = 5,     /* whole-field device copies (resync of the scratch field) */
    LS_K_KINDS = 6
} ls_kernel_kind;

typedef struct ls_ctx ls_ctx;

const char* ls_status_str(ls_status s);
/* Text of the last CUDA error seen by this process' libls (static storage; "" if none). */
const char* ls_last_cuda_error(void);

/* Create a context for an nx*ny*nz grid of `dtype` on the CURRENT CUDA device.
 * `cuda_stream` is a cudaStream_t (CUstream) handle cast to void*; NULL = the legacy default stream.
 * The ctx owns: per-brick flags and mask words, the T/N/U brick lists, counters, and (allocated on
 * first use by ls_step / ls_reinit*) one scratch field of nx*ny*nz elements.  Any n* >= 1 is
 * accepted (partial bricks at the high ends). */
ls_status ls_create(int32_t nx, int32_t ny, int32_t nz, ls_dtype dtype, void* cuda_stream, ls_ctx** out);
ls_status ls_destroy(ls_ctx* ctx);

/* Step 1: tubes T = {|phi| < gamma} (eq. 6) and N = T plus every in-domain
 * face neighbour of a T point (eq. 11; R6), as ascending lists of the 8^3 bricks that
 * hold at least one such point, each with its 512-bit mask.  Scans the whole grid.
 * `phi` is read only.  `dx` is accepted for symmetry with the paper's call and must be > 0; the
 * classification does not use it.  gamma = +inf puts every in-domain point in T.
 * The lists stay valid (inside the ctx) until the next ls_build_band / ls_step on this ctx. */
ls_status ls_build_band(ls_ctx* ctx, const void* phi, double dx, double gamma);

/* Counts of the band last built (by ls_build_band or the last step of ls_step).  Synchronises.
 * HOST out-pointers; any may be NULL. */
ls_status ls_band_counts(ls_ctx* ctx, int64_t* nT_points, int64_t* nN_points, int32_t* nT_bricks,
                         int32_t* nN_bricks);

/* Copy the band last built to HOST buffers sized from ls_band_counts: ids[n*_bricks] and
 * masks[8*n*_bricks].  Any pointer may be NULL (that list is skipped).  Synchronises. */
ls_status ls_band_export(ls_ctx* ctx, int32_t* T_ids, uint64_t* T_masks, int32_t* N_ids, uint64_t* N_masks);

/* Step 2, eq. 3 with F -> c(phi) F (eq. 8), gradients eq. 4-5
 * (PAPER.md:30-35), cut-off eq. 7:
 *     out(x) = phi(x) - dt * ( c(phi(x)) * [max(F,0) grad+ + min(F,0) grad-] )   for x in T,
 *     out(x) = phi(x)                                                           elsewhere (R8).
 * Uses the band last built on this ctx (LS_ERR_STATE if none).  If beta and gamma are both +inf the
 * call is the full-domain update (c == 1, T = grid) and needs no band.  `out` must not alias `phi`
 * (Jacobi, R15).  On return (stream order) `out` is defined at EVERY point. */
ls_status ls_advance(ls_ctx* ctx, const void* phi, const void* F, double dt, double dx, double beta,
                     double gamma, void* out);

/* Step 3: `iters` Jacobi iterations of eq. 12 with S of eq. 13
 * (R9-R12) on the tube N last built, from d^0 = phi_bar; then eq. 10 at
 * every point (R14).  iters = 0: clamp only.  `d` (out) must not alias `phi_bar` (read only).
 * Uses the ctx scratch field as the second Jacobi buffer. */
ls_status ls_reinit(ls_ctx* ctx, void* d, const void* phi_bar, double dtau, double dx, double gamma,
                    int32_t iters);

/* Step 3 "solved to steady state" (R13): as ls_reinit, but stops at the first k that is
 * a multiple of check_every (>= 1) with r_k = max_{x in N} |d^k - d^{k-1}| < tol, or at max_iters
 * (then returns LS_NOT_CONVERGED; `d` is still the clamped d^{max_iters}).  Synchronises once per
 * check.  HOST out-pointers iters_done / residual (r of the last iteration run) may be NULL. */
ls_status ls_reinit_tol(ls_ctx* ctx, void* d, const void* phi_bar, double dtau, double dx, double gamma,
                        double tol, int32_t max_iters, int32_t check_every, int32_t* iters_done,
                        double* residual);

/* Steps 1-3, n_steps times, on the ctx stream with no host synchronisation inside:
 * build T,N from phi^n -> Advance on T -> p->iters x Reinit on the SAME N (R7) -> eq. 10.
 * `phi` is updated in place; on completion it holds phi^{n+n_steps} at every point with
 * |phi| <= gamma everywhere (the whole-grid clamp of eq. 10 / R14 runs once per call, after the first
 * step: afterwards points outside N already hold +-gamma).  `F` is read only and static (R17).
 * n_steps = 0 is a no-op. */
ls_status ls_step(ls_ctx* ctx, void* phi, const void* F, const ls_params* p, int32_t n_steps);

/* Same as ls_step with HOST buffers (pageable or pinned): copies phi and F to ctx-owned device
 * fields, runs n_steps, copies phi back, and synchronises.  The end-to-end entry point.
 * F is static (R17): F_host = NULL reuses the F that the last call with a non-NULL F_host left on the
 * device (LS_ERR_STATE if there was none), which saves a third of the transfer.
 * A call with n_steps == 1 on a field of at least 64 MiB runs as a pipeline of z-slabs: one step depends on
 * p->iters + 1 layers around a point (eq. 3-5, 11, 12), so each slab is stepped on a window with that many halo
 * layers (ctx-owned window buffers and a child ctx of the window's shape) while later slabs are still being
 * uploaded and earlier ones downloaded — host-to-device copy, kernels and device-to-host copy overlap on three
 * ctx-owned streams (pinned host memory makes the copies asynchronous; pageable works).  The result and the work
 * counters (ls_stats) are bit-identical to the unsliced call; after such a call the ctx holds no band
 * (ls_band_counts / ls_band_export / ls_advance return LS_ERR_STATE until the next build), and ls_profile_* does
 * not see the windows' kernels. */
ls_status ls_step_host(ls_ctx* ctx, void* phi_host, const void* F_host, const ls_params* p, int32_t n_steps);

/* m-step batching with snapshot return (the paper keeps m results on the device and
 * copies them back per host round trip; writing output is ~16 % of its serial run time;
 * SURVEY.md section 8(f) f-2).  Runs ls_step's Steps 1-3 n_steps times and returns a copy of phi after every
 * `every`-th step (every >= 1) to HOST memory: host_out receives floor(n_steps / every) fields of
 * nx*ny*nz elements back to back (pinned memory makes the copies asynchronous; pageable works).
 * Snapshot k is copied device-to-device into one of two ctx-owned slots on the ctx stream, and from the slot
 * to the host on a second, ctx-owned stream while the following steps compute (events order the two
 * streams both ways).  `phi` is updated in place as by ls_step.  Synchronises both streams before it
 * returns, also when a step or a copy fails (then the first error is returned).  HOST out-pointer n_written (may be
 * NULL) = number of snapshots written.
 * p->chained is honoured for the first step; the remaining steps are chained internally. */
ls_status ls_step_snapshots(ls_ctx* ctx, void* phi, const void* F, const ls_params* p, int32_t n_steps,
                            int32_t every, void* host_out, int32_t* n_written);

/* Which band kernels a ctx uses.  The tiled kernels (32 x 8 x 8 tiles staged in shared memory by producer warps) need
 * rows that are 16-byte multiples and 16-byte aligned fields; everything else takes the scalar kernels (one CTA per
 * brick, any shape).  Both give the same bits.  On a grid of fewer than min_cells points the scalar kernels are used
 * even where the tiled ones could run: a tiled launch needs ~12 us to fill its pipeline, more than a scalar launch takes
 * on a small band.  Default 4 000 000 (the measured crossover on a B200: 160^3); 0 = tiled wherever possible;
 * negative = restore the default.  Takes effect from the next band launch. */
ls_status ls_tile_threshold(ls_ctx* ctx, int64_t min_cells);

/* Work counters since ls_create / the last ls_stats_reset: band point updates
 * sum_steps(|T_s| + iters*|N_s|) (dense advance: nx*ny*nz per call), narrow-band steps done, and
 * kernels launched by this ctx.  HOST out-pointers, any may be NULL.  Synchronises. */
ls_status ls_stats(ls_ctx* ctx, int64_t* point_updates, int64_t* steps, int64_t* kernel_launches);
ls_status ls_stats_reset(ls_ctx* ctx);

/* Per-kernel device timing.  While enabled, every launch (or launch group, for LS_K_BAND) this ctx
 * enqueues is bracketed by two CUDA events on the ctx stream; ls_profile_read synchronises and returns
 * the summed elapsed time (milliseconds) and the number of bracketed launches of one ls_kernel_kind
 * since the last ls_profile_reset / enable.  HOST out-pointers, either may be NULL.  The events cost a
 * few microseconds per launch: headline timings are taken with profiling off. */
ls_status ls_profile_enable(ls_ctx* ctx, int32_t on);
ls_status ls_profile_read(ls_ctx* ctx, int32_t kind, double* ms_total, int64_t* launches);
ls_status ls_profile_reset(ls_ctx* ctx);

/* DIAGNOSTIC, not part of the path: device self-check of the fp32 arithmetic: the band kernels evaluate two points per lane with packed
 * FADD2 / FMUL2 / FFMA2 instructions and hand-sequenced correctly rounded sqrt / divide; this runs both
 * that path and the plain scalar IEEE path (eq. 3-8 and eq. 12-13) on `n` pairs of seeded random 7-point
 * stencils (band-like values, arbitrary bit patterns, zeros, flat patches) on the current device and
 * returns how many of the 6n results (reinit, band Advance, dense Advance) differ in any bit (NaN == NaN).  Must be 0.  Runs on `cuda_stream`
 * and synchronises it.  HOST out-pointer. */
ls_status ls_selftest_math(void* cuda_stream, uint64_t seed, int64_t n, double dx, double dt, double beta,
                           double gamma, int64_t* mismatches);

#ifdef __cplusplus
}
#endif
#endif /* LS_H_ */
