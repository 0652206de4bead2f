/* ens.h — C ABI of libens: an ensemble of independent few-body systems advanced on one B200 (sm_100a) in FP64.
 *
 * The library is the data-parallel hot path of Swarm-NG (arxiv 1208.1157; `P:L<n>` = PAPER.md line n):
 * the fixed-step 4th-order time-symmetrized Hermite integrator (Alg. 2; Eq. 3-4) and a
 * mixed-variable symplectic kick / Kepler-drift step, both inside the generic
 * integrator loop of Alg. 1 with fused stop monitors.  Readings of the garbled or
 * silent passages (R1..R15, R-M1..R-M7) are listed in DESIGN.md §3.
 *
 * Conventions
 *   - Every function returns an int: 0 = ENS_OK, < 0 = error.  No exception crosses this boundary.
 *   - Caller arrays are plain C-order FP64:  pos, vel [n_sys][n_body][3];  mass [n_sys][n_body];
 *     time, E [n_sys];  L [n_sys][3];  status int32 [n_sys];  nsteps int64 [n_sys].
 *     `memspace` says whether those pointers are HOST (pageable or pinned) or DEVICE (cudaMalloc'd, or the
 *     data_ptr of a torch CUDA tensor) addresses.  The caller owns them and keeps them alive until the
 *     call's work on `stream` has run.
 *   - The handle owns its internal structure-of-arrays device buffers (layout: DESIGN.md §5).
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Device-space calls only
 *     enqueue work and return: they never allocate (ens_create allocates everything ens_integrate needs).
 *     Host-space calls enqueue the copies on `stream` and then wait for it, so the host buffers are complete (get)
 *     or reusable (set) on return; the first one also allocates the device staging area, unless
 *     ens_reserve_host_staging did so before.
 *   - Work enqueued for ONE handle must be stream-ordered: use one stream per handle, or order the streams yourself
 *     (the handle's state rows, work counters and staging are shared by its calls).  Different handles are independent
 *     and may run concurrently on different streams.
 *   - Every call runs on the CUDA device that was current when the handle was created, whatever device is current
 *     in the calling thread, and leaves the caller's current device unchanged.  Pointers and streams passed to a
 *     call must belong to that device.
 *   - Body 0 is the central body.  G = 1.  No softening.
 *   - There is no CPU fallback: without a CUDA device every compute call returns ENS_ECUDA.
 */
#ifndef ENS_H
#define ENS_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define ENS_API __attribute__((visibility("default")))
#else
#define ENS_API
#endif

typedef struct ens ens_t; /* opaque */

enum {
    ENS_OK = 0, ENS_EINVAL = -1, ENS_ENOMEM = -2, ENS_ECUDA = -3, ENS_ESTATE = -4, ENS_EUNSUPPORTED = -5,
    ENS_ETOOLARGE = -6 /* ens_hermite_static: the ensemble needs more than the library's static scratch holds */
};
enum {
    ENS_HERMITE = 0, ENS_MVS = 1, ENS_HERMITE_ADAPTIVE = 2, ENS_HERMITE_CARRY = 3, ENS_RKCK = 4,
    ENS_MVS_MERGED = 5,    /* MVS with the adjacent half sub-steps of consecutive steps merged */
    ENS_RKCK_ADAPTIVE = 6  /* Cash-Karp with step rejection and step-size control (R-RK2') */
};
enum { ENS_HOST = 0, ENS_DEVICE = 1 };
/* per-system status (Alg. 1 "state").  DONE_* become ACTIVE again at the next ens_integrate;
 * STOP_* are sticky until ens_set_state. */
enum {
    ENS_ACTIVE = 0,
    ENS_DONE_TIME = 1,      /* t reached t_end (reading R10: stop when t >= t_end, last step not clipped) */
    ENS_DONE_STEPS = 2,     /* max_steps taken in this call (Alg. 1 max-iterations) */
    ENS_STOP_CLOSE = 3,     /* some pair separation < r_close after a step (monitor; R11) */
    ENS_STOP_EJECT = 4,     /* some body farther than r_eject from the coordinate origin after a step (R11) */
    ENS_STOP_NONFINITE = 5, /* a position became non-finite */
    ENS_STOP_STEPSIZE = 6   /* adaptive Runge-Kutta: the rejected step shrank until t + h == t (tolerance unreachable) */
};

/* Create an ensemble of n_sys >= 1 systems of 2 <= n_body <= 16 bodies on the current CUDA device and
 * allocate its device buffers.  *out receives the handle.  EINVAL: bad sizes or out == NULL.
 * ENOMEM: allocation failed.  ECUDA: no device / CUDA error. */
ENS_API int ens_create(int64_t n_sys, int n_body, ens_t **out);

/* Free the handle and its buffers (synchronises the device first).  NULL is a no-op returning ENS_OK. */
ENS_API int ens_destroy(ens_t *e);

/* Allocate the device staging area the host-space calls copy through (n_sys * (7 n_body + 4) doubles) now instead
 * of inside the first host-space call.  Idempotent.  EINVAL: NULL handle.  ENOMEM. */
ENS_API int ens_reserve_host_staging(ens_t *e);

/* Load the state of every system (Alg. 1 "load initial configuration onto the GPU"; the only
 * bulk host->device transfer).  time == NULL means t = 0 for all.  Resets status to ACTIVE and
 * nsteps to 0.  Transposes the caller's [sys][body][3] arrays into the internal SoA layout on the device.
 * EINVAL: NULL e/pos/vel/mass or bad memspace. */
ENS_API int ens_set_state(ens_t *e, const double *pos, const double *vel, const double *mass, const double *time,
                  int memspace, void *stream);

/* Stop monitors evaluated after every step on the new state (Alg. 1 execute(M); thresholds from
 * BASELINE.json).  r_close <= 0 disables the close-approach monitor; r_eject = +inf (or <= 0) disables the
 * ejection monitor.  Strict inequalities: stop if r < r_close, or |x_i| > r_eject.  Default: both disabled.
 * EINVAL: NULL handle or NaN. */
ENS_API int ens_set_monitors(ens_t *e, double r_close, double r_eject);

/* Accuracy parameter eps of ENS_RKCK_ADAPTIVE ("user specified accuracy parameter"; default 1e-9): a trial step
 * is accepted when max(max|err_x| / (eps X), max|err_v| / (eps V)) <= 1.1, X and V the largest body distance and speed
 * of the system at the start of the step.  EINVAL: NULL handle, eps <= 0 or non-finite. */
ENS_API int ens_set_rk_tolerance(ens_t *e, double eps);

/* Rejected trial steps per system since ens_set_state (ENS_RKCK_ADAPTIVE), int64 [n_sys].  ESTATE: no state. */
ENS_API int ens_get_rejected(const ens_t *e, int64_t *nreject, int memspace, void *stream);

/* Advance every system independently (Alg. 1), entirely on the device, in ONE kernel launch
 * with the state resident in registers across all steps:
 *     while status == ACTIVE && steps_this_call < max_steps && time left:  step(dt); t += dt; ++nsteps; monitors
 * "time left" is direction aware: dt > 0: t < t_end;  dt < 0: t > t_end.  Use t_end = +inf (dt > 0) or -inf
 * (dt < 0) for pure step-count control.  integrator: ENS_HERMITE = predictor + 2 corrector iterations with 3
 * acceleration-and-jerk evaluations per step (Alg. 2; R3-R6); ENS_MVS = democratic-heliocentric
 * half-drift / half-kick / Kepler drift / half-kick / half-drift (R-M1..R-M7), which needs body 0
 * to dominate the mass; ENS_HERMITE_ADAPTIVE = the same Hermite step with the time step recomputed at the start of
 * every step from Eq. 5, step = dt [ sum_i |j_i|^2 / |a_i|^2 ]^(-1/2) over all bodies of the system
 * (R-A1, R-A2): here `dt` is the dimensionless step size scale tau (its sign gives the direction), every system
 * takes its own steps, and `time` advances by the step actually taken; ENS_HERMITE_CARRY = Alg. 2 exactly as printed
 * (reading R6-alt): fixed step, TWO evaluations per step, a^(0), j^(0) of a step being the a^(2), j^(2)
 * the previous step left behind (only the first step of a call evaluates at the state itself, so a run split over
 * two calls is not bit-identical to the unsplit one); ENS_RKCK = fixed-step Runge-Kutta Cash-Karp (P:L93-97,
 * P:L246-248): six acceleration evaluations per step, no jerk, the fifth-order solution propagated (R-RK1);
 * ENS_MVS_MERGED = the MVS map with the closing half drift / half kick of a step and the opening ones of the next
 * merged into a full kick and a full drift (the same map in exact arithmetic; rounding-level differences from ENS_MVS;
 * a run split over two calls closes and re-opens the half sub-steps); ENS_RKCK_ADAPTIVE = Cash-Karp with the embedded
 * error estimate controlling the step (reading R-RK2' of DESIGN.md section 3: the GSL manual's standard
 * control, step factors floor(16 f)/16): `dt` is the first trial step of every system (its sign gives the direction),
 * ens_set_rk_tolerance gives the accuracy parameter eps, a trial step whose error level exceeds 1.1 is rejected (state
 * and time untouched, counted in ens_get_rejected) and retried with a smaller step, `max_steps` counts accepted steps,
 * and a system whose step shrinks until t + h == t stops with ENS_STOP_STEPSIZE.
 * EINVAL: NULL handle, unknown integrator, dt == 0 or non-finite, NaN t_end, max_steps < 0.
 * ESTATE: no state was set.  ECUDA: launch failed. */
ENS_API int ens_integrate(ens_t *e, int integrator, double dt, double t_end, int64_t max_steps, void *stream);

/* Copy the state out (transposing back to [sys][body][3]).  Any out pointer may be NULL (skipped).
 * ESTATE: no state was set. */
ENS_API int ens_get_state(const ens_t *e, double *pos, double *vel, double *time, int32_t *status, int64_t *nsteps,
                  int memspace, void *stream);

/* ---- state log (the "log" action of the paper's monitors; readings R-L1, R-L2 of DESIGN.md) ---------- */
enum { ENS_LOG_SNAPSHOTS = 1, /* every system that advanced, after every segment */
       ENS_LOG_STOPS = 2      /* systems a stop monitor halted (status >= ENS_STOP_CLOSE), once, with their stop state */ };

/* Allocate (capacity > 0) or free (capacity == 0) the device log buffer of `capacity` records and empty it.  A
 * record is (system index, its total step count, its time, its status, pos [n_body][3], vel [n_body][3]).  Waits for
 * `stream` first.  EINVAL: NULL handle or capacity < 0.  ENOMEM. */
ENS_API int ens_log_enable(ens_t *e, int64_t capacity, void *stream);

/* ens_integrate in segments of `log_every` steps; after each segment a kernel on the same stream appends one record
 * for every system selected by `what` (ENS_LOG_* bits) that advanced since its last record.  Everything is enqueued:
 * no host round trip between segments.  Records beyond the capacity are dropped and counted.  Results are
 * bit-identical to one ens_integrate of max_steps for ENS_HERMITE, ENS_HERMITE_ADAPTIVE, ENS_RKCK and ENS_MVS up to
 * its coordinate round trip (their step is a pure function of the state); ENS_HERMITE_CARRY re-evaluates at every
 * segment start.  EINVAL: as ens_integrate, or log_every < 1, or no ENS_LOG_* bit, or more than 10^6 segments
 * (max_steps / log_every: every segment is enqueued from the host whether or not systems still run).
 * ESTATE: no log buffer / state. */
ENS_API int ens_integrate_logged(ens_t *e, int integrator, double dt, double t_end, int64_t max_steps,
                                 int64_t log_every, int what, void *stream);

/* Copy up to max_records records out, in the order they were appended (within one segment: unspecified).
 * *n_records = records copied, *n_dropped (may be NULL) = records lost to the capacity.  Any array pointer may be
 * NULL.  Always waits for `stream` (the count is a host value).  ESTATE: no log buffer. */
ENS_API int ens_log_read(const ens_t *e, int64_t *n_records, int64_t *n_dropped, int64_t *sys, int64_t *nsteps,
                         double *time, int32_t *status, double *pos, double *vel, int64_t max_records, int memspace,
                         void *stream);

/* Total energy E = sum 1/2 m v^2 - sum_{i<k} m_i m_k / r_ik (Eq. 6, each pair once: R9) and, if
 * L != NULL, total angular momentum sum m x cross v, per system, computed on the device ("only 1-4 values
 * per system need to be transferred").  EINVAL: NULL e or E.  ESTATE: no state was set. */
ENS_API int ens_energy(const ens_t *e, double *E, double *L, int memspace, void *stream);

/* The fixed-step Hermite step loop of ens_integrate(ENS_HERMITE) WITHOUT A HANDLE AND WITHOUT ANY ALLOCATION, for
 * callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it):
 * no cudaMalloc, cudaFree or allocating library routine is called, here or in anything this calls.
 * The caller owns the ensemble, as DEVICE arrays in the library's structure-of-arrays layout, all
 * advanced in place:  pos, vel [n_body * 3][n_pad] (row = body * 3 + component, n_pad >= n_sys consecutive systems
 * per row);  mass [n_body][n_pad] (read only);  time [n_pad];  status int32 [n_pad] (ENS_ACTIVE = 0 to start a system;
 * the status semantics of ens_integrate: DONE_* run again, STOP_* are skipped);  nsteps int64 [n_pad] (the steps
 * taken are ADDED to it).  Columns n_sys .. n_pad - 1 are never touched.  dt, t_end, max_steps as in ens_integrate;
 * r_close, r_eject as in ens_set_monitors (<= 0 switches that monitor off).  Results are bit-identical to
 * ens_integrate(ENS_HERMITE) on the same state (the step is a pure function of the state, reading R6).
 * The kernel is the time-sliced persistent grid; its scratch (a task counter and one int32
 * progress word per warp-group of 32 / L systems, L = lanes per system: 1 for n_body <= 8, 3 or 5 above) is a
 * file-scope device array of ENS_STATIC_MAX_GROUPS words + 256 bytes = 256.25 KB that every GPU which loads the
 * library holds until the process exits.  Limit: ceil(n_sys / (32 / L)) <= ENS_STATIC_MAX_GROUPS, i.e. at most
 * 2097152 systems of n_body <= 8, 655360 of 9..12 bodies (393216 of 10), 393216 of 13..16; beyond it ETOOLARGE.
 * ALL calls on one device share that array and each finds the last call's contents in it: the words a launch uses are
 * cleared on `stream` right before its kernel, so calls ordered on one stream (or by events) are safe, and two calls
 * that OVERLAP on the GPU race on it (undefined results).  The first call on a device looks the array's device
 * address up (cudaGetSymbolAddress, with that device current) and loads the module: make it outside graph capture.
 * Runs on the CURRENT device; only enqueues on `stream` and returns.
 * EINVAL: NULL pointer, n_sys < 1, n_pad < n_sys, n_body outside 2..16, dt == 0 or non-finite, NaN t_end / r_close /
 * r_eject, max_steps < 0.  ETOOLARGE: see above.  ECUDA: no device / lookup or launch failed. */
#define ENS_STATIC_MAX_GROUPS 65536
ENS_API int ens_hermite_static(double *pos, double *vel, const double *mass, double *time, int32_t *status,
                               int64_t *nsteps, int64_t n_sys, int64_t n_pad, int n_body, double dt, double t_end,
                               int64_t max_steps, double r_close, double r_eject, void *stream);

/* Static description of an error code; for ENS_ECUDA the text of the last CUDA error seen by this thread. */
ENS_API const char *ens_strerror(int code);

/* ---- measurement helpers (not part of the method; used by bench.py and the tests) -------------------- */

/* Sizes the library chose for this handle: out[0] = padded system count of the SoA rows, out[1] = lanes
 * per system L, out[2] = bodies per lane B, out[3] = threads per block, out[4] = blocks of the last or next
 * step-loop launch, out[5] = registers per thread of that kernel, out[6] = resident blocks per SM (occupancy
 * API), out[7] = number of kernels this handle has launched so far, out[8] = local-memory (stack / spill) bytes per
 * thread of that kernel, out[9] = 1 if the last fixed-step Hermite launch ran on the time-sliced persistent grid. */
ENS_API int ens_get_info(const ens_t *e, int64_t out[10]);

/* Time (ms, CUDA events on `stream`) the last ens_integrate kernel took; waits for it to finish.
 * ESTATE if nothing was launched. */
ENS_API int ens_last_kernel_ms(const ens_t *e, float *ms);

/* FP64 pipe microbenchmark: every thread of a full-occupancy grid runs `iters` rounds of 8 independent
 * dependent-DFMA chains.  *lane_fma_per_s receives FP64 lane-FMA/s (CUDA-event timed on `stream`), the
 * measured denominator of the FP64 roofline (MEASURED_PEAKS.json has no FP64 entry). */
ENS_API int ens_fp64_peak(int64_t iters, double *lane_fma_per_s, void *stream);

/* Device function test hook: y[i] = the library's FP64 reciprocal square root of x[i] (MUFU.RSQ64H seed +
 * FP64 refinement, P:L276 / R14), device pointers, n elements. */
ENS_API int ens_test_rsqrt(const double *x, double *y, int64_t n, void *stream);

/* Device function test hook: y[i] = the library's FP64 reciprocal of x[i] (MUFU.RCP64H seed + FP64 refinement; used
 * by the MVS Kepler drift instead of the IEEE divide), device pointers, n elements. */
ENS_API int ens_test_rcp(const double *x, double *y, int64_t n, void *stream);

/* Test / measurement hook: override a launch-time choice of the library for this handle (value 0 = back to the
 * library's default).  Results never depend on these (tests/test_gpu_hermite.py checks bit-identity); they exist for
 * the sweeps recorded in DESIGN.md section 8.  EINVAL: NULL handle, unknown option, value out of range. */
enum {
    ENS_OPT_THREADS = 0,            /* threads per block of the step-loop kernels (multiple of 32, <= the kernel's bound) */
    ENS_OPT_ADAPTIVE_UNORDERED = 1, /* 1: adaptive kernels hand systems out in index order (no longest-first pre-pass) */
    ENS_OPT_SLICE_MODE = 2,         /* fixed-step Hermite: 0 library decides, 1 always time-sliced grid, 2 never */
    ENS_OPT_SLICE_STEPS = 3,        /* steps per time slice */
    ENS_OPT_SLICE_WARPS_PER_SM = 4  /* persistent warps per SM of the time-sliced grid (<= what fits) */
};
ENS_API int ens_test_set_option(ens_t *e, int option, int64_t value);

#ifdef __cplusplus
}
#endif
#endif /* ENS_H */
