/*
 * aig.h -- C ABI of libaig: B200-native (sm_100a) atom-ion trajectory integrator.
 *
 * Hot path of arxiv/paper_2509_12381 ("GPU-Accelerated MATLAB Software for Atom-Ion
 * Dynamics"): integrate N independent 12-component atom-ion trajectories (PAPER.md:69,
 * eq. (3)-(10) at :71-90) with the adaptive Dormand-Prince 5(4) Runge-Kutta scheme behind
 * MATLAB's ode45, keeping only the final state and a few scalar
 * observables computed on the fly, then bin the observables on the
 * device ("their distributions").
 *
 * Conventions
 *   - plain C, no torch / C++ types; every pointer is marked HOST or DEVICE;
 *   - all quantities in atomic units, FP64; counters int32; flags uint8;
 *   - state layout: row k (0-based) of y0 / y_final is the paper's y_{k+1}:
 *     rows 0-2 ion position, 3-5 ion velocity, 6-8 atom position, 9-11 atom velocity;
 *     SoA: element (k, i) at offset k*N + i;
 *   - the caller owns every buffer; nothing allocated by the library outlives a call
 *     (aig_run_host frees what it allocates before returning);
 *   - work is enqueued on `cuda_stream` (a cudaStream_t passed as void*, NULL = default
 *     stream); no host synchronisation inside unless stated; outputs are valid once the
 *     stream has synchronised;
 *   - return value: 0 = AIG_OK, negative = error (see aig_strerror).  Numerical failure of one
 *     trajectory is NOT an error return: it is reported in status[i].
 *   - there is no CPU fallback: without a CUDA device every compute call returns
 *     AIG_ERR_CUDA.
 */
#ifndef AIG_H_
#define AIG_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define AIG_VERSION 100 /* 0.1.0 */

/* error codes */
#define AIG_OK 0
#define AIG_ERR_NULL (-1)      /* required pointer is NULL */
#define AIG_ERR_SIZE (-2)      /* N < 0, N too large, bad bin count */
#define AIG_ERR_TOL (-3)       /* rtol <= 0, atol < 0, non-finite tolerances */
#define AIG_ERR_TIME (-4)      /* t_max <= t0 or non-finite */
#define AIG_ERR_PARAM (-5)     /* masses <= 0, max_steps < 1, non-finite parameter */
#define AIG_ERR_ALIGN (-6)     /* device pointer not aligned to its element size */
#define AIG_ERR_CUDA (-7)      /* CUDA runtime error (no device, launch failure, out of memory) */
#define AIG_ERR_STATIC_LIMIT (-8) /* aig_outliers_static only: N is beyond what its built-in scratch is stated for */

/* status[i] of one trajectory */
#define AIG_STATUS_EXIT 0      /* r > r_exit after the first radial minimum */
#define AIG_STATUS_TMAX 1      /* reached t_max */
#define AIG_STATUS_MAXSTEPS 2  /* max_steps accepted steps */
#define AIG_STATUS_FAILED 3    /* step size underflow / non-finite error estimate */

/* Physical and stop parameters shared by all trajectories of a call (HOST struct).
 * The paper replicates every constant N times as a gpuArray; here they are
 * kernel arguments (constant bank). */
typedef struct aig_params {
    double m_ion, m_atom; /* masses */
    double C4, C8;        /* V(r) = C8/r^8 - C4/r^4 */
    double a[3], q[3];    /* the PAPER'S per-axis trap convention, eq. (4)-(6):
                             acc_k = -(a_k + 2 q_k cos(Omega t)) * Omega^2/4 * x_k  (ion only) */
    double omega_rf;      /* Omega_rf; with a = q = 0 the trap is off */
    double t0;            /* start time = RF phase origin */
    double r_exit;        /* stop when r > r_exit after the first radial minimum; <= 0 disables */
    double r_turn;        /* a radial minimum counts as a turning point only if r < r_turn;
                             +inf counts all of them */
    int64_t max_steps;    /* accepted-step cap, paper default 1,000,000 */
    int32_t n_att, n_rep; /* NEXT-1: general exponents V(r) = -C_n/r^n + C_m/r^m with
                             n = n_att, C_n = C4, m = n_rep, C_m = C8, 1 <= n < m <= 32; 0, 0 = the
                             benchmark potential n = 4, m = 8.  Other pairs take a general force
                             routine (integer powers by repeated squaring, a square root when an
                             exponent is odd) and the natural work-queue order unless n = 4. */
} aig_params;

/* Per-trajectory outputs: caller-allocated DEVICE buffers, each of length N
 * (y_final: 12*N, SoA like y0; x_turn1: 3*N).  No pointer except x_turn1 may be NULL. */
typedef struct aig_out {
    double *y_final;       /* state at the last accepted step end (PAPER.md:192 yend1..12) */
    double *t_final;       /* time of that step end (tend) */
    double *lifetime;      /* t(last turning point) - t(first), 0 if fewer than two */
    double *angle;         /* angle in [0, pi] between initial and final atom velocity */
    double *r_min;         /* smallest atom-ion distance seen at t0 and accepted step ends */
    int32_t *n_acc;        /* accepted steps ("nsteps") */
    int32_t *n_rej;        /* failed attempts */
    int32_t *n_turn;       /* counted inner turning points ("bounces") */
    int32_t *status;       /* AIG_STATUS_* */
    uint8_t *complex_flag; /* 1 if n_turn >= 2 (one bounce = simple) */
    double *x_turn1;       /* OPTIONAL (NULL = not recorded), [3][N] SoA: ion position at the accepted step end
                              that counted the first turning point -- the paper's "position" observable is its
                              norm ("how far the ion is from the origin during the first bounce", PAPER.md:495;
                              DESIGN.md reading S29); NaN for a trajectory with n_turn = 0 */
} aig_out;

/* Bin edges of the observable histograms: DEVICE pointers to strictly increasing doubles
 * (n_bins + 1 of them).  Bin j holds edges[j] <= v < edges[j+1].  Each bin count is in 1 .. 2048
 * (AIG_ERR_SIZE otherwise; aig_run_host checks the same). */
typedef struct aig_hist_spec {
    const double *angle_edges;
    int32_t n_angle_bins;
    const double *life_edges;
    int32_t n_life_bins;
    int32_t n_turn_bins; /* n_turn is clamped to n_turn_bins - 1 */
} aig_hist_spec;

/* Histogram outputs: DEVICE uint64 arrays, ACCUMULATED into (the caller zeroes them):
 *   angle    [n_angle_bins + 2]: [0] underflow, [1 + j] bin j, [n + 1] overflow and NaN
 *   lifetime [n_life_bins + 2] : same layout, over trajectories with complex_flag = 1 only
 *   n_turn   [n_turn_bins], status [4]
 *   totals   [4]: sum n_acc, sum n_rej, number of complexes, number of trajectories */
typedef struct aig_hist {
    uint64_t *angle, *lifetime, *n_turn, *status, *totals;
} aig_hist;

/* Bytes of DEVICE scratch aig_integrate needs for N trajectories: 256 uint64 counters (work
 * queues, slot counts, a stage timeline), the work-queue order (one int64 and one class byte per trajectory) and
 * min(N, max(2^20, N/4)) checkpoint slots of 224 B for suspended trajectories. */
size_t aig_workspace_bytes(int64_t N);

/* Integrate N trajectories from t0 to the first stop (exit radius, t_max, max_steps).
 *   p         HOST   parameters (copied into the launch)
 *   y0        DEVICE [12][N] initial conditions, never written
 *   t_max     end of the time span (> p->t0);  rtol > 0, atol >= 0: ode45 tolerances
 *   out       HOST struct of DEVICE pointers
 *   workspace DEVICE scratch of >= aig_workspace_bytes(N) bytes, 8-byte aligned
 * Persistent kernels: each thread integrates one trajectory at a time and refills from a
 * global work queue when it finishes (PAPER.md:186-202 runs one array element per thread);
 * trajectories that outlive a step budget (long-lived complexes) are handed, while the bulk is
 * still running, to a second kernel that spreads one trajectory over six lanes on SMs of its own
 * (an internal second stream, joined to `cuda_stream` before the call's work is complete from
 * the caller's point of view).  Every result is bit-identical whichever kernel produced it.
 * Thread safety: may be called concurrently from several host threads (different streams and
 * workspaces); the enqueue section is serialised per process, and calls that overlap on one
 * device share the internal stream, so their six-lane passes run one after the other.
 * p->max_steps must fit the int32 step counters (<= 2^31 - 1), else AIG_ERR_PARAM. */
int aig_integrate(const aig_params *p, const double *y0, int64_t N, double t_max, double rtol,
                  double atol, const aig_out *out, void *workspace, void *cuda_stream);

/* Reduce the observables of N trajectories into histograms and totals (PAPER.md:23, :457,
 * :517; the paper does this on the host after gather()).  obs: HOST struct of DEVICE
 * pointers as written by aig_integrate (uses angle, lifetime, n_acc, n_rej, n_turn, status,
 * complex_flag); spec: HOST struct of DEVICE edge pointers; out: HOST struct of DEVICE
 * pointers. */
int aig_histogram(const aig_out *obs, int64_t N, const aig_hist_spec *spec, const aig_hist *out,
                  void *cuda_stream);

/* ---- NEXT-1: the paper's remaining observables and its outliers ------------------ */

/* Observables of PAPER.md:495-497 that follow from the initial and final states (and, for
 * `position`, from aig_out.x_turn1): DEVICE arrays of length N, written by aig_observables.  The
 * paper names them without formulas; the readings are DESIGN.md S24-S26, S29:
 *   dist      "the final atom-ion distance"          |x_atom - x_ion| at the end
 *   KE        "the final kinetic energy of the ion"  m_ion |v_ion|^2 / 2
 *   transfer  "the momentum transfered by the atom"  m_atom |v_atom(end) - v_atom(t0)|
 *   position  "how far the ion is from the origin    |x_turn1|, NaN without a bounce; OPTIONAL (NULL =
 *              during the first bounce"               skipped), needs out->x_turn1 of aig_integrate     */
typedef struct aig_obs_extra {
    double *dist, *KE, *transfer;
    double *position;
} aig_obs_extra;

/* dist, KE, transfer (and position) of N trajectories from y0 (DEVICE [12][N]) and out->y_final as
 * written by aig_integrate (only y_final, and x_turn1 when extra->position is set, are read).  One
 * HBM-bound kernel on `cuda_stream`. */
int aig_observables(const aig_params *p, const double *y0, const aig_out *out, int64_t N,
                    const aig_obs_extra *extra, void *cuda_stream);

/* "outliers" (the trajectories with the highest and lowest value of each
 * observable): result (DEVICE int64 [8][2]) receives, for the observables
 *   0 angle, 1 n_turn ("bounces"), 2 lifetime, 3 transfer, 4 dist, 5 n_acc ("nsteps"), 6 KE, 7 position
 * the index of the smallest ([k][0]) and of the largest ([k][1]) value; the smallest index wins a
 * tie, NaNs are skipped (trajectories without a bounce have no position), -1 when nothing qualifies
 * (N = 0, or extra->position = NULL for row 7).  One pass over the eight arrays.
 * workspace: DEVICE scratch of aig_outliers_workspace_bytes() bytes, 16-byte aligned. */
size_t aig_outliers_workspace_bytes(void);
int aig_outliers(const aig_out *out, const aig_obs_extra *extra, int64_t N, int64_t *result,
                 void *workspace, void *cuda_stream);

/* ---- aig_outliers without a workspace: for callers that must not allocate device memory -------------
 * Some users of this library run where device memory is not theirs to ask for: an analysis hook inside a
 * long ensemble run whose host program handed out all of the GPU's memory at start-up and wants no
 * cudaMalloc afterwards (it synchronises the whole device and can fail hours into a run), a plug-in of a
 * framework that owns the allocator, a service with a fixed memory plan.  They can pass the observable
 * arrays they already hold and an [8][2] result, but have nowhere to take aig_outliers' workspace from.
 * aig_outliers_static is aig_outliers (same kernel, same result rows, same tie and NaN rules,
 * PAPER.md:521) with the scratch -- one ticket counter and the per-block partial extrema -- kept in an
 * array that is part of the library itself: AIG_OUTLIERS_STATIC_SCRATCH_BYTES (131,328) bytes of device
 * memory on every GPU that loads libaig, held until the process exits, enough for a grid of 512 blocks.
 *   - The call itself allocates and frees nothing (no cudaMalloc / cudaFree, no library routine that
 *     does); it enqueues one 256-byte memset and one kernel on `cuda_stream`.
 *   - Limit: N <= AIG_OUTLIERS_STATIC_MAX_N (2^28 trajectories, 64 times the largest ensemble of
 *     BASELINE.json); a larger N returns AIG_ERR_STATIC_LIMIT before anything touches the device -- use
 *     aig_outliers with a workspace of your own for that.  N = 0 is valid (every row -1, -1).
 *   - The first call on each device looks up the array's device address (once per device, with that device
 *     current, kept afterwards).  Make that first call outside any stream capture.
 *   - All calls on a device share the one array, and it keeps what the previous call left in it; each call
 *     zeroes the counter it needs, in stream order.  Two calls whose kernels can overlap on the GPU
 *     (different streams, or different host threads on different streams) race on it and give wrong
 *     indices: keep calls on one device in one stream order.  aig_outliers has no such restriction.
 * out, extra, result: as for aig_outliers (HOST structs of DEVICE pointers; result DEVICE int64 [8][2]). */
#define AIG_OUTLIERS_STATIC_MAX_N (1LL << 28)
#define AIG_OUTLIERS_STATIC_SCRATCH_BYTES 131328
int64_t aig_outliers_static_max_n(void);
int aig_outliers_static(const aig_out *out, const aig_obs_extra *extra, int64_t N, int64_t *result,
                        void *cuda_stream);

/* ---- NEXT-3: replay of one trajectory, every accepted step recorded ---------------
 * the paper simulates its longest-lived (or a custom) trajectory again "with
 * the same exact initial conditions" to display it.  y0: DEVICE [12], one state in the paper's
 * component order.  Row j (j < cap) of the record is the state after accepted step j + 1:
 * t_out[j], y_out[k * cap + j] (SoA like y_final).  The integration always runs to its stop;
 * steps beyond `cap` are not recorded.  n_out: DEVICE int64 [4] = accepted steps, status
 * (AIG_STATUS_*), failed attempts, counted turning points.  One thread, the arithmetic of
 * aig_integrate: the last recorded row equals that call's y_final for the same y0 bit for bit.
 * Data only: no plotting (out of scope). */
int aig_trace(const aig_params *p, const double *y0, double t_max, double rtol, double atol,
              int64_t cap, double *t_out, double *y_out, int64_t *n_out, void *cuda_stream);

/* Test hook: ONE attempted DP5(4) step of size h[i] from (t[i], y[:, i]) for each of N
 * states.  DEVICE: y [12][N], t [N], h [N], ynew [12][N] (5th-order solution), err [N]
 * (ode45's scaled error estimate; the step would be accepted iff err <= rtol). */
int aig_step_once(const aig_params *p, const double *y, const double *t, const double *h,
                  int64_t N, double rtol, double atol, double *ynew, double *err,
                  void *cuda_stream);

/* End-to-end convenience entry with HOST buffers: allocates device memory, copies y0 to the
 * device, runs aig_integrate (+ aig_histogram when hist_spec/hist_out are non-NULL, with
 * HOST edge pointers and HOST uint64 outputs, zeroed by the call), copies every non-NULL
 * member of `out` (HOST pointers here) back, frees the device memory and synchronises.
 * Blocking. */
int aig_run_host(const aig_params *p, const double *y0_host, int64_t N, double t_max, double rtol,
                 double atol, const aig_out *out_host, const aig_hist_spec *hist_spec_host,
                 const aig_hist *hist_out_host);

/* NEXT-2: an observable against the launch direction (the paper's heatmaps, PAPER.md:483, :517:
 * "as a function of the spherical angles theta and phi", the "(theta, phi) for the initial conditions of the atom").
 * The direction of trajectory i is that of the ATOM's position at t0, rows 6-8 of y0 alone (about the trap centre; a
 * thermally displaced ion does not shift the cells): u = (1 - cos theta)/2 in [0, 1] (equal steps of u are equal solid
 * angles, eq. (12)-(13) at PAPER.md:92-98) and phi = atan2(y, x) brought into [phi_edges[0], phi_edges[0] + 2 pi), so a
 * window may straddle phi = 0 (edges from -0.5 to 0.5, say); the edges must span at most one turn.  Cells are given by
 * explicit edges (DEVICE pointers, strictly increasing, n + 1 of them, n in 1..4096 each): cell (a, b) holds
 * u_edges[a] <= u < u_edges[a+1], phi_edges[b] <= phi < phi_edges[b+1].  For every trajectory inside the window whose
 * value is not NaN: count[a * n_phi + b] += 1, sum[a * n_phi + b] += value[i] (DEVICE arrays of n_u * n_phi,
 * ACCUMULATED into: the caller zeroes them; sum / count is the map).  An atom AT the origin has no direction and is
 * skipped.  At a pole (theta = 0 or pi) phi is undefined and read as 0: on a "uniform" grid whose theta window
 * starts at 0 (the paper's default octant) the nphi trajectories of that row are one and the same launch point and all
 * land in the cell that holds phi = 0.  Such a grid is index-ordered (i = theta index * nphi + phi index), so its map
 * is simply the value array viewed as [ntheta][nphi], which is what the paper does; aig_map2d is for "random"
 * positions and for re-binning.  Away from the poles, with edges half-way between the grid directions, the map of a
 * grid workload equals that view (head-on or "thermal"). */
typedef struct aig_map_spec {
    const double *u_edges;
    int32_t n_u;
    const double *phi_edges;
    int32_t n_phi;
} aig_map_spec;
int aig_map2d(const double *y0, int64_t N, const double *value, const aig_map_spec *spec, uint64_t *count,
              double *sum, void *cuda_stream);

/* The potential front-end of the paper's parameter block (the form V(r) = -C_n/r^n + C_m/r^m at :51):
 * the user gives two of the four numbers C_n, C_m, D_e (well depth, Hartree), R_e (equilibrium distance, Bohr) and
 * "the code then analytically calculates" the others from V'(R_e) = 0 and V(R_e) = -D_e.  HOST arithmetic, no
 * device, no allocation.  mode / meaning of (a, b):
 *   AIG_POT_CNCM  a = C_n, b = C_m   ("CnCm": both constants known; D_e and R_e follow)
 *   AIG_POT_CNDE  a = C_n, b = D_e   ("CnDe": C_m and R_e follow)
 *   AIG_POT_DERE  a = D_e, b = R_e   ("DeRe": C_n and C_m follow)
 * All four values are written (the two given ones are copied through); an output pointer may be NULL.  The result
 * goes into aig_params as C4 = C_n, C8 = C_m, n_att = n, n_rep = m.  AIG_ERR_PARAM unless 1 <= n < m <= 32 and a, b
 * are finite and > 0; AIG_ERR_SIZE for an unknown mode.  The paper's listing (n = 4, m = 8,
 * C_n = 159.5455, D_e = 1 K) prints C_m = 2.00949488627505397797e+09 and R_e = 70.8448174250339519631. */
#define AIG_POT_CNCM 0
#define AIG_POT_CNDE 1
#define AIG_POT_DERE 2
int aig_potential(int mode, int n, int m, double a, double b, double *Cn, double *Cm, double *De, double *Re);

/* Measurement aid: run a register-resident FP64 FMA chain kernel on every SM and return the
 * achieved non-tensor FP64 rate in FLOP/s through *flops_per_s (blocking; used by bench.py as
 * the measured ALU roofline denominator). ilp in [1, 16] independent chains per thread. */
int aig_fp64_peak_probe(int iters, int ilp, double *flops_per_s, double *elapsed_ms);

/* Launch geometry the integrator would use on the current device (for reporting):
 * writes SM count, resident blocks per SM, threads per block, registers per thread and
 * local-memory (spill) bytes per thread of the RF-trap integrator kernel. */
int aig_kernel_info(int *sm_count, int *blocks_per_sm, int *threads_per_block,
                    int *regs_per_thread, int *local_bytes_per_thread);

/* Number of CUDA kernels libaig has launched in this process so far (integrator, histogram and
 * step-once kernels; the FP64 probe is not counted).  bench.py reports the difference over its
 * timed region as "gpu_launches". */
uint64_t aig_kernel_launches(void);

/* Test / tuning hook: the schedule aig_integrate uses from now on in this process.
 *   tail_iters  iterations a warp of the per-thread integrator keeps stepping after its work
 *               queue ran dry before it hands its trajectories over (default 1024)
 *   budget      accepted steps after which a trajectory is offered to the six-lane integrator
 *               (default 2048)
 *   split_sms   SMs the six-lane pass owns while the bulk pass runs beside it (12)
 *   split_grid  one-warp blocks per SM of the final six-lane pass (8)
 *   plan        0: natural order; 1: three classes, slow capture candidates first (default)
 *   kappa       candidates are trajectories with impact parameter < kappa Langevin radii (1.5)
 * Scheduling never changes a result (tests/test_gpu_parity.py::test_schedule_invariance).
 * Returns AIG_ERR_PARAM for out-of-range values.  Not thread-safe against concurrent
 * aig_integrate calls that should see the old schedule.  The library reads no environment
 * variable: these two calls are the only way to change the schedule. */
int aig_set_schedule(int tail_iters, int budget, int split_sms, int split_grid, int plan, double kappa);

/* All knobs of the schedule (the six above and the finer ones). */
typedef struct aig_schedule {
    int32_t tail_iters, budget, split_sms, split_grid, plan;
    double kappa;
    int32_t depth;        /* budget hand-overs pause while this many published slots wait to be taken (64) */
    int32_t mean_factor;  /* ... and are only for trajectories this many times longer than the mean of the
                             finished ones (4; 0 = the plain budget) */
    int32_t drain_lanes;  /* queue empty: a warp hands over what it still runs once this few lanes are alive (10) */
    double slow0, slow1;  /* class 0: candidates with u^2 < slow0 <u^2> (0.5); class 1 also takes anything
                             with u^2 < slow1 <u^2> (0.1) */
    int32_t refill_batch, refill_wait; /* idle lanes of a warp that trigger its refill (8), or iterations
                                          one of them has waited (16) */
    int32_t poll_iters;   /* six-lane warps with idle groups look for new slots every this many iterations (32) */
    int32_t hist_blocks_per_sm; /* grid of aig_histogram's kernel: blocks of 256 threads per SM (8) */
} aig_schedule;
/* s = NULL restores the defaults.  AIG_ERR_PARAM for out-of-range values. */
int aig_set_schedule_ex(const aig_schedule *s);
int aig_get_schedule(aig_schedule *s);

const char *aig_strerror(int code);
int aig_version(void);

#ifdef __cplusplus
}
#endif
#endif /* AIG_H_ */
