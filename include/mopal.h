/*
 * mopal.h - C ABI of libmopal: the data-parallel hot path of Mercury-Opal's
 * (arxiv 2601.19654) fully interacting n-body integration on one B200 (sm_100a).
 *
 * What the library computes (citations are /root/reference/PAPER.md lines; the
 * paper elides all arithmetic in <...> placeholders, so each operation is the
 * reading recorded in DESIGN.md section 3):
 *
 *   mo_accel      force block LOOP 2:
 *                   a_i = sum_{j != i} gm_j K_ij (x_j - x_i) / r_ij^3,
 *                   K_ij = changeover weight of r_ij with rc = max(rcrit_i, rcrit_j)
 *                   (critical radius, PAPER.md:104 fn. 14); body-body terms only.
 *   mo_drift      keplerian drift of every body about the star, mu = G m_star, over dt
 *                   by Gauss f,g in universal variables (arxes_drift, PAPER.md:59,
 *                   130, 231-233; iflag -> MO_ENOCONV).
 *   mo_encounters mce_snif: per-body x,y extremes over the step
 *                   padded by rcrit (LOOP 1-2), then for every i<j: boxes overlap and
 *                   estimated minimum separation over the step <= max(rcrit_i,rcrit_j)
 *                   (LOOP 3) -> pair list (ice/jce), per-body flag (ce), count (nce).
 *   mo_step       mdt_hy (Fig. 1, 202-226): kick h/2, stellar jump h/2,
 *                   copy x0,v0, drift h, encounter check, jump h/2, accel, kick h/2 -
 *                   all state resident in HBM (the paper moves 7N doubles H<->D twice
 *                   per step).  By default no restore and no
 *                   Bulirsch-Stoer resolution of flagged pairs; mo_set_resolve switches the
 *                   on-device resolution (the paper's host-side mdt_hkce) in.
 *
 * Units: AU, day, Msun; gm = G * mass.  Coordinates are democratic heliocentric:
 * heliocentric positions, barycentric velocities (PAPER.md:84, 100 fn. 12).
 * Bodies are indexed 0..nb-1; the star (the paper's array element 1,
 * PAPER.md:134) is not a body, only m_star.
 *
 * Layout: every per-body 3-vector array is SoA, 3 planes of `ld` doubles:
 * component c of body b at [c*ld + b]; ld >= nb, ld % 4 == 0, base 16-byte aligned.
 *
 * Memory: "device" pointers are CUDA device memory of the current device,
 * "host" pointers ordinary (preferably pinned) host memory.  The CALLER owns every
 * array passed in; the context BORROWS the device arrays given to mo_create for its
 * whole lifetime and owns only its scratch (freed by mo_destroy).
 *
 * Execution: all work is enqueued on the stream given to mo_create and the calls
 * return immediately, except where a host out-pointer is given (then the call
 * synchronises that stream before returning).  No exceptions, abort, exit or
 * stdout; failures are return codes.  Asynchronous CUDA errors surface as
 * MO_ECUDA on the next synchronising call.  There is no CPU fallback: without a
 * CUDA device mo_create returns MO_ECUDA.
 *
 * Environment (read once, at mo_create / mo_set_nbig; everything else is a function
 * argument): MO_DEBUG=1 synchronises after every launch so that a failing kernel is
 * reported by the call that launched it.  Five switches exist for the test-suite only -
 * they force a kernel that the problem size alone would not select, so that every kernel
 * is checked at sizes the oracle handles: MO_PSM=0 (no lane-split pair kernel), MO_SYM=1
 * (two-sided pair kernel at any size), MO_SYM_CH=n (its j tiles per work unit), MO_SMALL=0 /
 * MO_SMALL_MAX=n (single-CTA front end off / up to n bodies).  They change which kernel
 * computes a result, never the result's definition.
 */
#ifndef MOPAL_H
#define MOPAL_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mo_ctx mo_ctx; /* opaque */

typedef enum {
    MO_OK = 0,
    MO_EINVAL = 1,    /* null / misaligned pointer, nb < 1, ld < nb or ld % 4, non-finite or
                         non-positive m_star / G, dt == 0 or non-finite, cap < 0, nsteps < 0 */
    MO_ENOMEM = 2,    /* scratch allocation failed */
    MO_ECUDA = 3,     /* CUDA runtime error (or no device) */
    MO_EOVERFLOW = 4, /* more encounter pairs than `cap`: the first `cap` pairs in sorted
                         order are stored, the count is still the true total */
    MO_ENOCONV = 5,   /* >= 1 body's Kepler solve failed (paper's iflag);
                         those bodies are left unchanged, the others advanced */
    MO_ERESOLVE = 6,  /* mo_set_resolve / mo_resolve: >= 1 encounter component was not resolved (no
                         convergence, or a truncated pair list); its bodies kept the Kepler-drift
                         result of that step.  Sticky: counted in mo_stats.resolve_fail */
    MO_ELIMIT = 7     /* mo_accel_static: nb beyond mo_accel_static_max_nb() - its scratch is a fixed
                         array, there is no allocation to fall back to.  Nothing was launched */
} mo_status;

typedef struct {
    int64_t steps_done; /* mo_step steps completed since mo_create */
    int64_t nce_last;   /* encounter pairs found by the last encounter pass (true total) */
    int64_t nce_total;  /* sum of nce_last over all passes */
    int32_t drift_fail; /* bodies whose Kepler solve failed, cumulative */
    int32_t max_newton; /* largest Newton iteration count any body needed so far */
    int32_t resolve_fail; /* encounter components the Bulirsch-Stoer solve gave up on, cumulative */
    int32_t reserved;
} mo_stats;

/* Create a context.  Reads `mass` once (gm = G*mass is kept in scratch).
 *   nb       number of bodies (>= 1); ld plane stride in doubles
 *   m_star,G central mass (Msun) and gravitational constant (AU^3 Msun^-1 day^-2;
 *            Mercury's units give G = k^2 = 2.959122082855911e-4)
 *   mass     device, nb           (borrowed only during the call)
 *   x, v     device, 3*ld each    (borrowed, read and written)
 *   a        device, 3*ld         (borrowed, written by mo_accel / mo_step)
 *   rcrit    device, nb, AU       (borrowed; read at every launch, so the caller may
 *                                  update it between calls as the paper does)
 *   pairs    device, 2*cap int32  (borrowed, out) pair k = (pairs[2k], pairs[2k+1]), 0-based,
 *                                  i<j, sorted by i then j; may be NULL iff cap == 0
 *   flag     device, nb uint8     (borrowed, out) 1 iff the body is in a flagged pair
 *   cuda_stream  cudaStream_t; NULL = legacy default stream                          */
mo_status mo_create(mo_ctx **out, int32_t nb, int32_t ld, double m_star, double G,
                    const double *mass, double *x, double *v, double *a,
                    const double *rcrit, int32_t *pairs, int64_t cap, uint8_t *flag,
                    void *cuda_stream);

/* a <- accel(x).  Asynchronous. */
mo_status mo_accel(mo_ctx *ctx);

/* x, v <- Kepler drift over dt (dt may be negative).  Asynchronous; failures are
 * counted in stats.drift_fail and reported by the next synchronising call. */
mo_status mo_drift(mo_ctx *ctx, double dt);

/* Encounter check for a step of size dt that took (x0, v0) to the context's current
 * (x, v).  x0, v0: device, 3*ld, or both NULL to use the snapshot the last mo_step (or
 * mo_snapshot) stored.  Writes pairs / flag; if count_host != NULL the stream is
 * synchronised and *count_host receives the true pair count (MO_EOVERFLOW if > cap). */
mo_status mo_encounters(mo_ctx *ctx, double dt, const double *x0, const double *v0,
                        int64_t *count_host);

/* nsteps hybrid steps of size dt.  `a` must be current for `x` unless the context has
 * never computed it or mo_invalidate_accel was called (then it is computed first, the
 * paper's first-call logic).  stats_host nullable; if given the call
 * synchronises and returns MO_EOVERFLOW / MO_ENOCONV / MO_ERESOLVE (in that order of
 * precedence) if any of them happened since mo_create. */
mo_status mo_step(mo_ctx *ctx, double dt, int32_t nsteps, mo_stats *stats_host);

void mo_destroy(mo_ctx *ctx);

/* ---- extras ------------------------------------------------------------- */

/* Big x all variant (the paper's own loop bounds): bodies
 * 0..nbig-1 are the "big" bodies.  Only they are gravity sources (mo_accel: a_i = sum over
 * j < nbig, j != i, for every body i), only their boxes are padded by rcrit, and only they can
 * be the first member of an encounter pair (i < nbig, i < j < nb).  Kick, stellar jump
 * (P = sum over ALL bodies of gm v), snapshot and drift still run over every body.
 * nbig = nb (the default after mo_create) is the fully interacting case.  1 <= nbig <= nb, else
 * MO_EINVAL.  Changing nbig drops the cached step graph and the pair-kernel scratch and
 * invalidates `a`.  Synchronises the stream. */
mo_status mo_set_nbig(mo_ctx *ctx, int32_t nbig);

/* ---- per-step support routines on the device (readings H-1..H-4, E-1..E-3) ---
 * The paper names these next to the hot path and runs them on the host, copying the critical
 * radii to the device every step (PAPER.md:291 item 3); here they stay on the device. */

/* mco_h2dh / mce_dh2h (PAPER.md:84 item 1, fn. 12).  In place on v (positions are heliocentric in
 * both systems).  mo_h2dh: heliocentric -> barycentric velocities, v_j -= sum m v / (m_star + sum m);
 * mo_dh2h: the inverse, v_j += sum m v / m_star.  Asynchronous on the context's stream. */
mo_status mo_h2dh(mo_ctx *ctx);
mo_status mo_dh2h(mo_ctx *ctx);

/* mce_hill + critical radius (PAPER.md:87, 94 fn. 13-14, 291).  Overwrites the caller's rcrit array
 * (device, nb doubles - the array given to mo_create, now written by the library) with
 * n_hill * r_H, r_H = d * (m / (3 m_star))^(1/3); mode 0: d = |x_j|, the instantaneous star-planet
 * separation; mode 1: d = osculating semi-major axis from x and the heliocentric velocity (unbound
 * bodies: |x_j|).  rhill_dev (nullable, device, nb doubles) receives r_H.  x heliocentric, v
 * barycentric.  MO_EINVAL: n_hill not finite or < 0, mode not 0/1.  Asynchronous. */
mo_status mo_hill(mo_ctx *ctx, double n_hill, int32_t mode, double *rhill_dev);

/* Make mo_step run mo_hill(n_hill, mode) at the start of every step ("the mce_hill routine is
 * called at each timestep"): encounters and the closing accelerations of step n use
 * the radii of the positions at the start of step n.  mode -1 switches it off (the default).
 * Drops the cached step graph. */
mo_status mo_set_hill(mo_ctx *ctx, double n_hill, int32_t mode);

/* mxx_en: kinetic energy T (star included), star-body potential Us, body-body potential
 * Up over the interacting pairs (i < j, i < nbig), E = T + Us + Up, and the total angular momentum L,
 * all in the barycentric frame, Msun AU^2 day^-2 and Msun AU^2 day^-1.  Synchronises the stream.
 * O(nbig * nb) pair evaluations. */
typedef struct { double T, Us, Up, E, L[3]; } mo_energy_t;
mo_status mo_energy(mo_ctx *ctx, mo_energy_t *out_host);

/* ---- close-encounter resolution on the device (the paper's host-side mdt_hkce, PAPER.md:104 fn. 14,
 * 126, 297-315; readings X-1..X-5) -------------------------------------------------------------
 * The bodies of the current encounter pair list (the last mo_encounters / mo_step) are restored to the
 * snapshot x0, v0 and integrated over dt with a Bulirsch-Stoer scheme (modified midpoint, 2..16 substeps,
 * polynomial extrapolation) whose local error stays below tol relative to |x_i|, |v_i| of every body, under
 * the star's Kepler term and the (1 - K)-weighted forces of the listed pairs - the complement of the
 * K-weighted kick; x, v of those bodies (which must hold the Kepler-drift result of the other bodies) are
 * overwritten.  Each connected component of the pair graph is its own system with its own step control; a
 * massless body (mass 0: the test particles of the big x all regime) exerts no force and is integrated in a
 * small system of its own with its massive partners.  Components of any size are resolved (up to 1023 pairs
 * in shared memory, one thread per body; larger ones streamed through global scratch).  Without convergence
 * (40 rejected steps in a row), or when the pair list was truncated (count > cap), the bodies keep the
 * Kepler-drift result, the component is counted in mo_resolve_stats / mo_stats.resolve_fail and the next
 * synchronising call returns MO_ERESOLVE.  The result is deterministic (fixed summation orders).
 * Asynchronous.  MO_EINVAL: tol <= 0, dt == 0, no snapshot. */
mo_status mo_resolve(mo_ctx *ctx, double dt, double tol);
/* Make mo_step resolve the encounters of every step (between the encounter check and the second jump,
 * PAPER.md:297-315); tol <= 0 switches it off (the default).  Drops the cached step graph. */
mo_status mo_set_resolve(mo_ctx *ctx, double tol);
/* Last resolution: out4 = {bodies integrated and written back, accepted BS steps and right-hand-side
 * evaluations summed over the systems, systems not resolved}.  Synchronises. */
mo_status mo_resolve_stats(mo_ctx *ctx, int32_t *out4);

/* ---- the pair sum sharded over several GPUs (the paper sees MPI over CPU clusters as
 * the only multi-device route) -----------------------------------------------------------------------
 * One process and one context per GPU, all holding the WHOLE state (identical arrays on every rank).  Only the
 * O(N^2) pair sum is split: after mo_set_shard(rank, world) a context evaluates its contiguous share of the pair
 * kernel's work units (two-sided kernel, nb > 2560: units of the triangle, so a rank's result is a PARTIAL
 * acceleration of every body; big x all mode: blocks of bodies i, the other rows 0), and the caller sums `a` over the
 * ranks (one all-reduce of 3*ld doubles per step, e.g. NCCL through torch.distributed - the library itself holds no
 * communicator).  Every O(N) stage and the encounter pass run replicated on every rank, on identical data, so the
 * states stay bit-identical across the ranks.  Protocol:
 *     mo_accel(ctx); <sum a over ranks>; mo_accel_summed(ctx);
 *     per step: mo_step_begin(ctx, dt); <sum a over ranks>; mo_step_end(ctx, dt, stats);
 * mo_step itself returns MO_EINVAL while world > 1.  MO_EINVAL also for sizes whose pair kernel does not split
 * (fully interacting systems of up to 2560 bodies: a step there is tens of microseconds). */
mo_status mo_set_shard(mo_ctx *ctx, int32_t rank, int32_t world);
/* [lo, hi) = rank's contiguous share of n work units: lo = n*rank/world, hi = n*(rank+1)/world.  Host only. */
mo_status mo_shard_range(int64_t n, int32_t rank, int32_t world, int64_t *lo, int64_t *hi);
/* The pair kernel's work units and this context's share of them (for inspection). */
mo_status mo_shard_units(const mo_ctx *ctx, int64_t *units, int64_t *lo, int64_t *hi);
/* kick, jump, snapshot, drift, encounter pass, jump, this rank's share of a(x).  Needs a summed a (see above). */
mo_status mo_step_begin(mo_ctx *ctx, double dt);
/* Tell the context that `a` now holds the sum over the ranks. */
mo_status mo_accel_summed(mo_ctx *ctx);
/* The closing kick v += dt/2 a with the summed a; stats_host as in mo_step (nullable; synchronises if given). */
mo_status mo_step_end(mo_ctx *ctx, double dt, mo_stats *stats_host);

/* Copy the current x, v into the context's x0, v0 snapshot (asynchronous). */
mo_status mo_snapshot(mo_ctx *ctx);
/* Device pointers of the snapshot planes (3*ld doubles each), for inspection. */
mo_status mo_snapshot_ptrs(mo_ctx *ctx, const double **x0, const double **v0);
/* Copy the snapshot into caller-owned device arrays (3*ld doubles each; asynchronous). */
mo_status mo_snapshot_copy(mo_ctx *ctx, double *x0_dst, double *v0_dst);
/* mce_snif LOOP 1-2, for inspection: copy the per-body boxes of the last encounter
 * pass (mo_encounters or the last mo_step) into box_dst (device, 4*nb doubles): body b at
 * box_dst[4b..4b+3] = {lo_x, hi_x, lo_y, hi_y}, extremes of the cubic Hermite interpolant over the step,
 * padded by rcrit for the big bodies.  Asynchronous.  MO_EINVAL before any encounter pass. */
mo_status mo_boxes_copy(mo_ctx *ctx, double *box_dst);
/* Tell the context that the caller changed x: the next mo_step recomputes a first. */
mo_status mo_invalidate_accel(mo_ctx *ctx);
/* Synchronise the stream and read the statistics. */
mo_status mo_get_stats(mo_ctx *ctx, mo_stats *stats_host);
/* Number of libmopal kernels launched on behalf of this context so far. */
int64_t mo_launch_count(const mo_ctx *ctx);
/* Bytes of device scratch the context owns so far.  The partial-sum buffers of the pair kernel
 * are allocated by the first mo_accel / mo_step (which may therefore return MO_ENOMEM). */
int64_t mo_workspace_bytes(const mo_ctx *ctx);

/* Host-buffer variant of the step (the paper's per-step data region):
 * copies x_host, v_host (3*ld each) and, if non-NULL, rcrit_host (nb) to the device,
 * runs nsteps steps, copies x, v back, and if pairs_host != NULL the first
 * min(count, cap_host, cap) pairs.  a_is_current != 0 asserts that the device-resident
 * `a` is valid for x_host (e.g. x_host is what the previous call returned); otherwise
 * it is recomputed first.  Always synchronises.  Writes the borrowed rcrit buffer. */
mo_status mo_step_host(mo_ctx *ctx, double dt, int32_t nsteps, double *x_host,
                       double *v_host, const double *rcrit_host, int32_t a_is_current,
                       int32_t *pairs_host, int64_t cap_host, mo_stats *stats_host);

/* Host-buffer variant of mo_accel: uploads x_host (3*ld), computes, downloads a_host
 * (3*ld).  Synchronises. */
mo_status mo_accel_host(mo_ctx *ctx, const double *x_host, double *a_host);

/* Measures the FP64 FMA issue peak of the current device with a register-resident
 * DFMA loop (148 SMs x 64 lanes x 2 flop x clock on B200): runs `reps` back-to-back timed
 * launches on `cuda_stream` and writes the best single launch's TFLOP/s (burst) and its
 * duration in ms, and - if tflops_mean_out != NULL - the TFLOP/s over the whole train of
 * launches (sustained, under the power cap when reps spans seconds).  Used as the measured
 * denominator of the pair kernel's roofline (MEASURED_PEAKS.json has no FP64 figure). */
mo_status mo_probe_fp64_peak(void *cuda_stream, int32_t reps, double *tflops_out,
                             double *ms_out, double *tflops_mean_out);

/* Pair-kernel launch geometry chosen for this nb: i-bodies per thread, j-splits,
 * CTAs, resident CTAs per SM (all nullable). */
mo_status mo_pair_geometry(const mo_ctx *ctx, int32_t *ipt, int32_t *jsplit,
                           int32_t *ctas, int32_t *ctas_per_sm);

/* Name of the pair kernel this context launches for mo_accel ("pair_sym_kernel": two-sided, nb > 2560
 * fully interacting; "pair_big_kernel": few gravity sources after mo_set_nbig; else "pair_accel_kernel").
 * Static string; NULL for a NULL context. */
const char *mo_pair_kernel_name(const mo_ctx *ctx);

/* Time of the last pair-accel kernel launch alone, measured with CUDA events on the
 * context's stream when timing was enabled with mo_set_kernel_timing(ctx, 1).
 * Synchronises.  ms_out receives the mean over the launches since enabling (and
 * n_out their number); both reset on read. */
mo_status mo_set_kernel_timing(mo_ctx *ctx, int32_t on);
mo_status mo_pair_kernel_ms(mo_ctx *ctx, double *ms_out, int32_t *n_out);

/* ---- No-allocation entry point -------------------------------------------------------------
 * mo_accel_static: a(x) of a fully interacting system - the same operation as mo_accel (force block
 * LOOP 2 with the changeover weight K; readings A-1..A-9), by the same
 * kernels (pack, two-sided pair sum with 2 bodies per lane, fixed-order reduce), for callers that cannot
 * call cudaMalloc: code under CUDA graph capture, tight serving loops, harnesses that forbid it.  It
 * needs no context and calls no cudaMalloc / cudaFree / allocating library routine, ever: the kernels'
 * scratch (packed tiles, work-unit list, row and column partial sums) is ONE file-scope device array of
 * 2.7 MB inside the library, which every GPU that loads the library holds until exit.
 *   nb            bodies, 1 <= nb <= mo_accel_static_max_nb() (4096); larger -> MO_ELIMIT, nothing launched
 *   ld            leading dimension of x and a (ld >= nb, ld % 4 == 0)
 *   gm, rcrit     device, nb doubles each: G m_j and the changeover radii (read)
 *   x             device, 3*ld doubles, SoA planes x | y | z, democratic-heliocentric positions (read)
 *   a             device, 3*ld doubles (written: rows < nb of each plane; nothing else is touched)
 *   cuda_stream   cudaStream_t; NULL = legacy default stream.  Four kernels are enqueued; asynchronous
 * All pointers 16-byte aligned, caller-owned.  The result equals mo_accel's to rounding (same arithmetic per
 * pair, a different fixed summation tree) and is bit-reproducible from call to call.
 * The array is looked up once per device (cudaGetSymbolAddress, with the caller's current device) and is
 * SHARED by every call on that device; it keeps the last call's contents, none of which a later call reads
 * before rewriting it (nothing has to start at zero).  Calls that overlap on the GPU - two streams, two
 * host threads, two captured graphs replayed side by side - RACE on it: serialise them (one stream, or
 * events).  Contexts (mo_create) do not use the array.
 * MO_EINVAL: nb < 1, ld < nb, ld % 4, null / misaligned pointer.  MO_ECUDA: no device / launch error. */
int32_t mo_accel_static_max_nb(void);
mo_status mo_accel_static(int32_t nb, int32_t ld, const double *gm, const double *x,
                          const double *rcrit, double *a, void *cuda_stream);

const char *mo_strerror(mo_status s);
const char *mo_version(void);

#ifdef __cplusplus
}
#endif
#endif /* MOPAL_H */
