/*
 * aig_oracle.c -- CPU ORACLE.  TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, single-threaded FP64 implementation of the hot path of
 * arxiv/paper_2509_12381 ("GPU-Accelerated MATLAB Software for Atom-Ion Dynamics"):
 * Dormand-Prince 5(4) adaptive Runge-Kutta ("the algorithm behind ode45",
 * PAPER.md:23, :43, :112-114, section 3) on the 12-component atom-ion ODE
 * (eq. (3)-(10)) with on-the-fly scalar observables.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may build, load or call this file.  It shares no code, header, table or constant
 * generator with the CUDA path (paper_2509_12381_b200/csrc/) and neither includes the
 * other.  Compile WITHOUT floating-point contraction (-ffp-contract=off): every
 * operation below is one IEEE-754 double operation, in the order written.
 *
 * The paper prints none of the solver's constants (Fig. 2 is an image, Fig. 6 is
 * missing); they are the published Dormand-Prince 1980 pair (paper ref. [5]) and the
 * ode45 default controller of Shampine-Reichelt 1997 (paper ref. [21]); every such
 * reading is listed in DESIGN.md ("Readings of the paper", S1-S23).
 *
 * Pins (tests/test_oracle_pins.py, all "-m not gpu"): rational order conditions of the
 * tableau, 5th-order convergence on y'=-y, one step against scipy.integrate.RK45 (same
 * published tableau, independent code), f(t,y) against finite differences of the
 * Hamiltonian eq. (1)-(2), exact free motion, the harmonic-trap closed form
 * (PAPER.md:432), Mathieu stability / secular frequency, two-body
 * conservation laws, the Langevin capture fraction, the classical deflection-angle
 * quadrature, and DOP853 cross-checks; the step-size controller (O3.3-O3.7: safety factors,
 * exponent, growth limit and its threshold, shrink floor, halving, kept step after a failure,
 * hmin = 16 ulp, last-step stretch, both ends of the step in the error scale) on the
 * quadrature problem y' = A t^4, where err = |A| (71/270000) h^5 / thr exactly and every step
 * sequence is computable by hand; lifetime / first / last bounce by a NumPy recomputation
 * from the replay record.  Parity UNPINNED pointwise for complex-forming (chaotic)
 * trajectories: ensemble statistics only.
 */
#include <math.h>
#include <stdint.h>
#include <stddef.h>
#include <string.h>

#define ORC_NMAX 16 /* largest ODE dimension the generic stepper accepts */

/* ---- parameters of one run (same field order as the product's aig_params, declared
 *      independently; all atomic units) ------------------------------------------------ */
typedef struct orc_params {
    double m_ion, m_atom;
    double C4, C8;        /* V(r) = -C4/r^4 + C8/r^8 */
    double a[3], q[3];    /* per-axis trap parameters, eq. (4)-(6) */
    double omega_rf;      /* Omega_rf; 0 => no trap */
    double t0;            /* start time = RF phase origin */
    double r_exit;        /* stop when r > r_exit after the first radial minimum; <= 0 disables */
    double r_turn;        /* a radial minimum is a counted turning point only if r < r_turn */
    int64_t max_steps;    /* accepted-step cap */
    int32_t n_att, n_rep; /* NEXT-1: V(r) = -C_n/r^n + C_m/r^m with n = n_att, C_n = C4,
                             m = n_rep, C_m = C8; 0, 0 = the benchmark potential n = 4, m = 8 */
} orc_params;

typedef void (*orc_rhs_fn)(double t, const double *y, double *f, int n, const void *ctx);
/* called after every accepted step with the step-end time and state; non-zero => stop */
typedef int (*orc_obs_fn)(double t_new, const double *y_new, void *obs);

/* ---- O2. Dormand-Prince 5(4) tableau (paper ref. [5]); 7 stages, FSAL --------------- */
static const double ORC_C[7] = {0.0, 1.0 / 5.0, 3.0 / 10.0, 4.0 / 5.0, 8.0 / 9.0, 1.0, 1.0};
static const double ORC_A[7][6] = {
    {0.0, 0.0, 0.0, 0.0, 0.0, 0.0},
    {1.0 / 5.0, 0.0, 0.0, 0.0, 0.0, 0.0},
    {3.0 / 40.0, 9.0 / 40.0, 0.0, 0.0, 0.0, 0.0},
    {44.0 / 45.0, -56.0 / 15.0, 32.0 / 9.0, 0.0, 0.0, 0.0},
    {19372.0 / 6561.0, -25360.0 / 2187.0, 64448.0 / 6561.0, -212.0 / 729.0, 0.0, 0.0},
    {9017.0 / 3168.0, -355.0 / 33.0, 46732.0 / 5247.0, 49.0 / 176.0, -5103.0 / 18656.0, 0.0},
    /* row 7 = the 5th-order weights b (FSAL) */
    {35.0 / 384.0, 0.0, 500.0 / 1113.0, 125.0 / 192.0, -2187.0 / 6784.0, 11.0 / 84.0}};
/* E = b - b*  (5th-order minus embedded 4th-order weights) */
static const double ORC_E[7] = {71.0 / 57600.0, 0.0, -71.0 / 16695.0, 71.0 / 1920.0,
                                -17253.0 / 339200.0, 22.0 / 525.0, -1.0 / 40.0};

/* expose the table so tests can check the order conditions on the doubles actually used */
void orc_tableau(double *c7, double *a7x6, double *e7)
{
    for (int s = 0; s < 7; ++s) {
        c7[s] = ORC_C[s];
        e7[s] = ORC_E[s];
        for (int j = 0; j < 6; ++j) a7x6[s * 6 + j] = ORC_A[s][j];
    }
}

/* ---- O1. force function f(t,y), eq. (3)-(10), written as printed ----- */
void orc_rhs_atomion(double t, const double *y, double *f, int n, const void *ctx)
{
    const orc_params *p = (const orc_params *)ctx;
    (void)n;
    const double dx = y[0] - y[6], dy = y[1] - y[7], dz = y[2] - y[8];
    const double r = sqrt(dx * dx + dy * dy + dz * dz);
    const double r2 = r * r, r4 = r2 * r2;
    const double r5 = r4 * r, r9 = r4 * r4 * r;
    double dVdr = 4.0 * p->C4 / r5 - 8.0 * p->C8 / r9;
    if (p->n_att != 0 || p->n_rep != 0) {
        /* general exponents: dV/dr = n C_n / r^(n+1) - m C_m / r^(m+1) */
        const double n = (double)p->n_att, m = (double)p->n_rep;
        dVdr = n * p->C4 / pow(r, n + 1.0) - m * p->C8 / pow(r, m + 1.0);
    }
    const double W2 = p->omega_rf * p->omega_rf / 4.0;
    const double cwt = cos(p->omega_rf * t);
    f[0] = y[3]; /* eq. (3) */
    f[1] = y[4];
    f[2] = y[5];
    f[3] = -1.0 / p->m_ion * dVdr * dx / r - (p->a[0] + 2.0 * p->q[0] * cwt) * W2 * y[0]; /* eq. (4) */
    f[4] = -1.0 / p->m_ion * dVdr * dy / r - (p->a[1] + 2.0 * p->q[1] * cwt) * W2 * y[1]; /* eq. (5) */
    f[5] = -1.0 / p->m_ion * dVdr * dz / r - (p->a[2] + 2.0 * p->q[2] * cwt) * W2 * y[2]; /* eq. (6) */
    f[6] = y[9]; /* eq. (7) */
    f[7] = y[10];
    f[8] = y[11];
    f[9] = -1.0 / p->m_atom * dVdr * (-dx) / r;  /* eq. (8): (y7 - y1) = -dx */
    f[10] = -1.0 / p->m_atom * dVdr * (-dy) / r; /* eq. (9) */
    f[11] = -1.0 / p->m_atom * dVdr * (-dz) / r; /* eq. (10) */
}

/* spacing of doubles above |t| (MATLAB eps(t)); hmin = 16*eps(t) in ode45 */
static double orc_ulp(double t)
{
    const double at = fabs(t);
    return nextafter(at, INFINITY) - at;
}

/* ---- O3.4  one attempted step ---------------------------------------------------------
 * k[0] must hold f(t, y).  Fills k[1..6], ynew (5th-order solution) and
 * err = h * max_i |sum_j E_j k_j,i| / max(|y_i|, |ynew_i|, thr)   (ode45's mixed norm). */
static void orc_dp45_attempt(orc_rhs_fn rhs, const void *ctx, int n, double t, const double *y,
                             double h, double t_new, double thr, double k[7][ORC_NMAX],
                             double *ynew, double *err)
{
    double ys[ORC_NMAX];
    for (int s = 1; s <= 6; ++s) {
        for (int i = 0; i < n; ++i) {
            double acc = 0.0;
            for (int j = 0; j < s; ++j) acc += (h * ORC_A[s][j]) * k[j][i];
            ys[i] = y[i] + acc;
        }
        /* stage 7 (s == 6) is evaluated at the step end and is next step's k1 (FSAL) */
        const double ts = (s == 6) ? t_new : t + ORC_C[s] * h;
        if (s == 6)
            for (int i = 0; i < n; ++i) ynew[i] = ys[i];
        rhs(ts, ys, k[s], n, ctx);
    }
    double emax = 0.0;
    int bad = 0;
    for (int i = 0; i < n; ++i) {
        double e = 0.0;
        for (int j = 0; j < 7; ++j) e += ORC_E[j] * k[j][i];
        const double sc = fmax(fmax(fabs(y[i]), fabs(ynew[i])), thr);
        const double ratio = fabs(e) / sc;
        if (ratio != ratio) bad = 1; /* NaN must not be dropped by fmax */
        emax = fmax(emax, ratio);
    }
    *err = bad ? NAN : h * emax;
}

/* one attempted step of size h from (t, y) for a generic right-hand side (test hook) */
int orc_dp45_step(orc_rhs_fn rhs, const void *ctx, int n, double t, const double *y, double h,
                  double rtol, double atol, double *ynew, double *err)
{
    if (n < 1 || n > ORC_NMAX || !(rtol > 0.0) || atol < 0.0) return -1;
    double k[7][ORC_NMAX];
    rhs(t, y, k[0], n, ctx);
    orc_dp45_attempt(rhs, ctx, n, t, y, h, t + h, atol / rtol, k, ynew, err);
    return 0;
}

/* ---- O3. the adaptive integration loop (ode45 defaults) -------------------------------
 * status: 0 stopped by the observer (exit radius), 1 reached t_max, 2 max_steps accepted
 * steps, 3 step-size underflow / non-finite error estimate.
 * Optional trace of accepted steps (t, y[n]) for tests and replay: trace_cap rows. */
int orc_dp45_integrate(orc_rhs_fn rhs, const void *ctx, int n, double t0, const double *y0,
                       double t_max, double rtol, double atol, int64_t max_steps,
                       orc_obs_fn observe, void *obs, double *y_final, double *t_final,
                       int64_t *n_acc_out, int64_t *n_rej_out, int *status_out,
                       double *trace_t, double *trace_y, int64_t trace_cap, int64_t *trace_len)
{
    if (n < 1 || n > ORC_NMAX || !(rtol > 0.0) || atol < 0.0 || !(t_max > t0)) return -1;
    double k[7][ORC_NMAX], y[ORC_NMAX], ynew[ORC_NMAX];
    const double thr = atol / rtol;       /* O3.1 */
    const double hmax = 0.1 * (t_max - t0);
    double t = t0;
    for (int i = 0; i < n; ++i) y[i] = y0[i];
    rhs(t, y, k[0], n, ctx);

    /* O3.2 initial step */
    double hmin = 16.0 * orc_ulp(t);
    double h = fmin(hmax, t_max - t0);
    double rho = 0.0;
    for (int i = 0; i < n; ++i) rho = fmax(rho, fabs(k[0][i]) / fmax(fabs(y[i]), thr));
    rho = rho / (0.8 * pow(rtol, 0.2));
    if (h * rho > 1.0) h = 1.0 / rho;
    h = fmax(h, hmin);

    int64_t n_acc = 0, n_rej = 0, n_tr = 0;
    int status = 3;
    for (;;) {
        /* O3.3 */
        hmin = 16.0 * orc_ulp(t);
        h = fmin(hmax, fmax(hmin, h));
        int last = 0;
        if (1.1 * h >= t_max - t) {
            h = t_max - t;
            last = 1;
        }
        int nofailed = 1, failed_hard = 0;
        double err = 0.0, t_new = t;
        for (;;) {
            t_new = last ? t_max : t + h; /* O3.4 */
            orc_dp45_attempt(rhs, ctx, n, t, y, h, t_new, thr, k, ynew, &err);
            if (err <= rtol) break;
            /* O3.5 failed attempt (NaN lands here too) */
            n_rej++;
            if (h <= hmin) {
                failed_hard = 1;
                break;
            }
            if (nofailed) {
                nofailed = 0;
                const double fac = (err == err) ? fmax(0.1, 0.8 * pow(rtol / err, 0.2)) : 0.1;
                h = fmax(hmin, h * fac);
            } else {
                h = fmax(hmin, 0.5 * h);
            }
            last = 0;
        }
        if (failed_hard) {
            status = 3;
            break;
        }
        /* O3.6 accepted */
        n_acc++;
        if (trace_t && n_tr < trace_cap) {
            trace_t[n_tr] = t_new;
            for (int i = 0; i < n; ++i) trace_y[n_tr * n + i] = ynew[i];
            n_tr++;
        }
        const int stop = observe ? observe(t_new, ynew, obs) : 0;
        if (stop || last || n_acc >= max_steps) {
            status = stop ? 0 : (last ? 1 : 2);
            t = t_new;
            for (int i = 0; i < n; ++i) y[i] = ynew[i];
            break;
        }
        /* O3.7 step-size update only after a step with no failed attempt */
        if (nofailed) {
            const double temp = 1.25 * pow(err / rtol, 0.2);
            if (temp > 0.2)
                h = h / temp;
            else
                h = 5.0 * h;
        }
        /* O3.8 advance; FSAL */
        t = t_new;
        for (int i = 0; i < n; ++i) {
            y[i] = ynew[i];
            k[0][i] = k[6][i];
        }
    }
    for (int i = 0; i < n; ++i) y_final[i] = y[i];
    *t_final = t;
    *n_acc_out = n_acc;
    *n_rej_out = n_rej;
    *status_out = status;
    if (trace_len) *trace_len = n_tr;
    return 0;
}

/* ---- O4. observables of one atom-ion trajectory ------------ */
typedef struct orc_obs_state {
    const orc_params *p;
    double s_prev; /* (r_atom - r_ion).(v_atom - v_ion) at the previous accepted step end */
    int any_min;   /* a radial minimum has been seen */
    int64_t n_turn;
    double t_first, t_last; /* times of the first / last counted turning point */
    double x_first[3];      /* ion position at the first counted turning point ("position") */
    double r_min;           /* min over t0 and accepted step ends of the atom-ion distance */
} orc_obs_state;

static void orc_rel(const double *y, double *r, double *s)
{
    const double dx = y[6] - y[0], dy = y[7] - y[1], dz = y[8] - y[2];
    const double ux = y[9] - y[3], uy = y[10] - y[4], uz = y[11] - y[5];
    *r = sqrt(dx * dx + dy * dy + dz * dz);
    *s = dx * ux + dy * uy + dz * uz;
}

static int orc_atomion_observe(double t_new, const double *y, void *o)
{
    orc_obs_state *st = (orc_obs_state *)o;
    double r, s;
    orc_rel(y, &r, &s);
    if (r < st->r_min) st->r_min = r;
    if (st->s_prev < 0.0 && s >= 0.0) { /* radial minimum: dr/dt changed sign - to + */
        st->any_min = 1;
        if (r < st->p->r_turn) {
            st->n_turn++;
            if (st->n_turn == 1) {
                st->t_first = t_new;
                for (int k = 0; k < 3; ++k) st->x_first[k] = y[k]; /* rows 0-2: ion position */
            }
            st->t_last = t_new;
        }
    }
    st->s_prev = s;
    /* exit radius: step-end test, no event location (reading S8) */
    if (st->p->r_exit > 0.0 && st->any_min && r > st->p->r_exit) return 1;
    return 0;
}

/* angle between two 3-vectors, in [0, pi]: atan2(|u x v|, u.v) (reading S12) */
static double orc_angle(const double *u, const double *v)
{
    const double cx = u[1] * v[2] - u[2] * v[1];
    const double cy = u[2] * v[0] - u[0] * v[2];
    const double cz = u[0] * v[1] - u[1] * v[0];
    const double dot = u[0] * v[0] + u[1] * v[1] + u[2] * v[2];
    return atan2(sqrt(cx * cx + cy * cy + cz * cz), dot);
}

/* ---- batch entry points on HOST SoA arrays, trajectories [i_begin, i_end) ----------- */
int orc_integrate(const orc_params *p, const double *y0 /* [12][N] */, int64_t N, double t_max,
                  double rtol, double atol, int64_t i_begin, int64_t i_end,
                  double *y_final /* [12][N] */, double *t_final, double *lifetime,
                  double *angle, double *r_min, int32_t *n_acc, int32_t *n_rej, int32_t *n_turn,
                  int32_t *status, uint8_t *complex_flag, double *x_turn1 /* [3][N] or NULL */)
{
    if (!p || !y0 || N < 0 || i_begin < 0 || i_end > N) return -1;
    if (!(rtol > 0.0) || atol < 0.0 || !(t_max > p->t0)) return -1;
    for (int64_t i = i_begin; i < i_end; ++i) {
        double y[12], yf[12], tf;
        for (int kk = 0; kk < 12; ++kk) y[kk] = y0[kk * N + i];
        orc_obs_state st;
        st.p = p;
        st.any_min = 0;
        st.n_turn = 0;
        st.t_first = 0.0;
        st.t_last = 0.0;
        st.x_first[0] = st.x_first[1] = st.x_first[2] = NAN; /* no bounce: no position (reading S29) */
        orc_rel(y, &st.r_min, &st.s_prev);
        int64_t na, nr;
        int stt;
        const int rc = orc_dp45_integrate(orc_rhs_atomion, p, 12, p->t0, y, t_max, rtol, atol,
                                          p->max_steps, orc_atomion_observe, &st, yf, &tf, &na,
                                          &nr, &stt, NULL, NULL, 0, NULL);
        if (rc) return rc;
        for (int kk = 0; kk < 12; ++kk) y_final[kk * N + i] = yf[kk];
        t_final[i] = tf;
        n_acc[i] = (int32_t)na;
        n_rej[i] = (int32_t)nr;
        n_turn[i] = (int32_t)st.n_turn;
        status[i] = stt;
        complex_flag[i] = (uint8_t)(st.n_turn >= 2);                 /* DESIGN.md reading S6 */
        lifetime[i] = (st.n_turn >= 2) ? st.t_last - st.t_first : 0.0;
        angle[i] = orc_angle(&y[9], &yf[9]); /* initial vs final atom velocity, lab frame */
        r_min[i] = st.r_min;
        if (x_turn1)
            for (int kk = 0; kk < 3; ++kk) x_turn1[kk * N + i] = st.x_first[kk];
    }
    return 0;
}

/* replay of ONE trajectory with every accepted step recorded (tests) */
int orc_integrate_trace(const orc_params *p, const double *y0 /* [12] */, double t_max,
                        double rtol, double atol, double *trace_t, double *trace_y /* [cap][12] */,
                        int64_t trace_cap, int64_t *trace_len, int *status)
{
    double yf[12], tf;
    int64_t na, nr;
    orc_obs_state st;
    st.p = p;
    st.any_min = 0;
    st.n_turn = 0;
    st.t_first = st.t_last = 0.0;
    st.x_first[0] = st.x_first[1] = st.x_first[2] = NAN;
    orc_rel(y0, &st.r_min, &st.s_prev);
    return orc_dp45_integrate(orc_rhs_atomion, p, 12, p->t0, y0, t_max, rtol, atol, p->max_steps,
                              orc_atomion_observe, &st, yf, &tf, &na, &nr, status, trace_t,
                              trace_y, trace_cap, trace_len);
}

/* one attempted step for N independent states (test hook mirrored by aig_step_once) */
int orc_step_once(const orc_params *p, const double *y /* [12][N] */, const double *t,
                  const double *h, int64_t N, double rtol, double atol,
                  double *ynew /* [12][N] */, double *err)
{
    if (!p || N < 0 || !(rtol > 0.0) || atol < 0.0) return -1;
    for (int64_t i = 0; i < N; ++i) {
        double yi[12], yn[12], e;
        for (int kk = 0; kk < 12; ++kk) yi[kk] = y[kk * N + i];
        const int rc = orc_dp45_step(orc_rhs_atomion, p, 12, t[i], yi, h[i], rtol, atol, yn, &e);
        if (rc) return rc;
        for (int kk = 0; kk < 12; ++kk) ynew[kk * N + i] = yn[kk];
        err[i] = e;
    }
    return 0;
}

/* f(t, y) for N states (pins of the force function) */
int orc_rhs_batch(const orc_params *p, const double *t, const double *y /* [12][N] */, int64_t N,
                  double *f /* [12][N] */)
{
    for (int64_t i = 0; i < N; ++i) {
        double yi[12], fi[12];
        for (int kk = 0; kk < 12; ++kk) yi[kk] = y[kk * N + i];
        orc_rhs_atomion(t[i], yi, fi, 12, p);
        for (int kk = 0; kk < 12; ++kk) f[kk * N + i] = fi[kk];
    }
    return 0;
}
