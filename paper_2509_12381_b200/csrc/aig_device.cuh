// aig_device.cuh -- device-side Dormand-Prince 5(4) stepper for the atom-ion ODE (sm_100a).
//
// What it computes: PAPER.md:71-90 (eq. (3)-(10)) integrated with the ode45 algorithm
// (constants: DESIGN.md "Integration loop").  How it computes it is
// B200-first and differs from the paper's seven pasted copies of f:
//   * the force depends on positions and time only, so the seven stages carry the six
//     ACCELERATION components only (Nystrom form, see gen_nystrom_tableau.py) -- 42 stage
//     doubles instead of 84, which is what lets a whole trajectory live in registers;
//   * (dV/dr)/r = 4 C4/r^6 - 8 C8/r^10 needs even powers of r only: no square root;
//   * cos(Omega t) is evaluated five times per attempt (c6 = c7 = 1 share one, k1 is FSAL);
//   * the error norm is a running maximum of ratios compared by cross-multiplication and
//     divided once; the controller's fifth root is a float seed + two Newton steps.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace aig {

#include "dp45_nystrom_tableau.inc"

enum TrapMode { TRAP_NONE = 0, TRAP_STATIC = 1, TRAP_RF = 2 };

// Derived constants of one call; passed by value as a kernel argument (constant bank).
struct KParams {
    double inv_mi, inv_ma;  // 1/m_ion, 1/m_atom
    double c4x4, c8x8;      // 4*C4, 8*C8
    double wa[3], wb[3];    // w_k(t) = wa_k + wb_k cos(Omega t): wa = a_k Om^2/4, wb = q_k Om^2/2
    double omega;
    double t0, t_max, hmax; // hmax = 0.1 (t_max - t0)
    double rtol, inv_rtol, thr;  // thr = atol/rtol
    double rho_scale;       // 1/(0.8 rtol^(1/5)) for the initial step
    double r_exit2, r_turn2;     // squared radii; r_exit2 = +inf disables the exit stop
    long long max_steps;
};

// (dV/dr)/r and the accelerations of both particles at positions (xi, xa), cos(Omega t) = cs.
// eq. (4)-(6): ion  acc_k = -(1/m_i)(dV/dr)(d_k/r) - w_k(t) x_k ;  eq. (8)-(10): atom acc_k = +(1/m_a)(dV/dr)(d_k/r)
// with d = x_ion - x_atom.
template <int TRAP>
__device__ __forceinline__ void accel(const KParams& P, double cs, const double (&xi)[3],
                                      const double (&xa)[3], double (&Ai)[3], double (&Aa)[3],
                                      double& r2_out)
{
    const double d0 = xi[0] - xa[0], d1 = xi[1] - xa[1], d2 = xi[2] - xa[2];
    const double r2 = fma(d2, d2, fma(d1, d1, d0 * d0));
    const double inv2 = 1.0 / r2;
    const double inv4 = inv2 * inv2;
    const double inv6 = inv4 * inv2;
    const double g = inv6 * fma(-P.c8x8, inv4, P.c4x4);  // 4C4/r^6 - 8C8/r^10
    const double ga = g * P.inv_ma;
    const double gi = -(g * P.inv_mi);
    Aa[0] = ga * d0;
    Aa[1] = ga * d1;
    Aa[2] = ga * d2;
    if (TRAP == TRAP_NONE) {
        Ai[0] = gi * d0;
        Ai[1] = gi * d1;
        Ai[2] = gi * d2;
    } else {
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const double w = (TRAP == TRAP_RF) ? fma(P.wb[k], cs, P.wa[k]) : P.wa[k];
            const double dk = (k == 0) ? d0 : (k == 1 ? d1 : d2);
            Ai[k] = fma(-w, xi[k], gi * dk);
        }
    }
    r2_out = r2;
}

// 16 * (spacing of doubles above |t|): ode45's hmin = 16 eps(t)
__device__ __forceinline__ double hmin_of(double t)
{
    const double at = fabs(t);
    const double up = __longlong_as_double(__double_as_longlong(at) + 1LL);
    return 16.0 * (up - at);
}

// q^(-1/5) for q > 0: float seed (MUFU lg2/ex2) + 2 Newton steps z <- z (1.2 - 0.2 q z^5);
// relative error ~1e-15.  q is clamped to [1e-30, 1e30] (the result is clamped by the caller).
__device__ __forceinline__ double inv_fifth_root(double q)
{
    q = fmin(fmax(q, 1e-30), 1e30);
    double z = (double)exp2f(-0.2f * __log2f((float)q));
    const double mq = -0.2 * q;
#pragma unroll
    for (int it = 0; it < 2; ++it) {
        const double z2 = z * z;
        const double z4 = z2 * z2;
        z = z * fma(mq, z4 * z, 1.2);
    }
    return z;
}

// Per-lane state of one trajectory (registers).
struct Traj {
    double xi[3], vi[3], xa[3], va[3];  // y at time t
    double Ai[3], Aa[3];                // accelerations at (t, y): stage 1, FSAL
    double t, h;
    double rmin2, sprev, t_first, t_last;
    int n_acc, n_rej, n_turn;
    bool any_min, last, nofailed;
};

// Result of one attempted step (before accept / reject).
struct Attempt {
    double xi[3], vi[3], xa[3], va[3];  // ynew
    double Ai[3], Aa[3];                // stage 7 = f(t_new, ynew) accelerations
    double t_new, err, r2, s;           // r2, s: |d|^2 and d.u at ynew (observables)
};

// One attempted Dormand-Prince step of size T.h from (T.t, y), stage 1 taken from T.Ai/T.Aa.
template <int TRAP>
__device__ __forceinline__ void dp45_attempt(const KParams& P, const Traj& T, Attempt& R)
{
    const double h = T.h;
    const double h2 = h * h;
    const double t_new = T.last ? P.t_max : T.t + h;

    // stage accelerations: A[l][0..2] ion, A[l][3..5] atom
    double A[7][6];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        A[0][k] = T.Ai[k];
        A[0][3 + k] = T.Aa[k];
    }
    const double x[6] = {T.xi[0], T.xi[1], T.xi[2], T.xa[0], T.xa[1], T.xa[2]};
    const double v[6] = {T.vi[0], T.vi[1], T.vi[2], T.va[0], T.va[1], T.va[2]};

    double r2 = 0.0;
    double xs[6];
#pragma unroll
    for (int s = 1; s <= 6; ++s) {
        const double hc = h * kC[s];
#pragma unroll
        for (int i = 0; i < 6; ++i) {
            double base = fma(hc, v[i], x[i]);
            if (s >= 2) {
                double acc = kAbar[s][0] * A[0][i];
#pragma unroll
                for (int l = 1; l <= s - 2; ++l) {
                    if (s == 6 && l == 1) continue;  // abar_72 = 0 exactly
                    acc = fma(kAbar[s][l], A[l][i], acc);
                }
                base = fma(h2, acc, base);
            }
            xs[i] = base;
        }
        double cs = 1.0;
        if (TRAP == TRAP_RF) cs = cos(P.omega * ((s >= 5) ? t_new : fma(kC[s], h, T.t)));
        const double sxi[3] = {xs[0], xs[1], xs[2]};
        const double sxa[3] = {xs[3], xs[4], xs[5]};
        double ai[3], aa[3];
        // stages 6 and 7 (c = 1) have different positions, so both are evaluated; they share cs
        accel<TRAP>(P, cs, sxi, sxa, ai, aa, r2);
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            A[s][k] = ai[k];
            A[s][3 + k] = aa[k];
        }
    }
    // xs now holds x_new (stage 7 position = 5th-order solution), A[6] = f(t_new, ynew)
    double vn[6], emax_n = 0.0, emax_d = 1.0;  // running max of ratios n/d
#pragma unroll
    for (int i = 0; i < 6; ++i) {
        // v_new = v + h sum b_l A_l   (b_2 = b_7 = 0)
        double sb = kB[0] * A[0][i];
        sb = fma(kB[2], A[2][i], sb);
        sb = fma(kB[3], A[3][i], sb);
        sb = fma(kB[4], A[4][i], sb);
        sb = fma(kB[5], A[5][i], sb);
        vn[i] = fma(h, sb, v[i]);
        // velocity rows of the error estimate: sum_l E_l A_l  (E_2 = 0)
        double ev = kE[0] * A[0][i];
        ev = fma(kE[2], A[2][i], ev);
        ev = fma(kE[3], A[3][i], ev);
        ev = fma(kE[4], A[4][i], ev);
        ev = fma(kE[5], A[5][i], ev);
        ev = fma(kE[6], A[6][i], ev);
        // position rows: h sum_l Ebar_l A_l  (Ebar_2 = Ebar_7 = 0)
        double ex = kEbar[0] * A[0][i];
        ex = fma(kEbar[2], A[2][i], ex);
        ex = fma(kEbar[3], A[3][i], ex);
        ex = fma(kEbar[4], A[4][i], ex);
        ex = fma(kEbar[5], A[5][i], ex);
        ex = ex * h;
        const double sv = fmax(fmax(fabs(v[i]), fabs(vn[i])), P.thr);
        const double sx = fmax(fmax(fabs(x[i]), fabs(xs[i])), P.thr);
        const double nv = fabs(ev), nx = fabs(ex);
        // n/d > emax_n/emax_d  <=>  n*emax_d > emax_n*d   (all denominators > 0)
        if (nv * emax_d > emax_n * sv) {
            emax_n = nv;
            emax_d = sv;
        }
        if (nx * emax_d > emax_n * sx) {
            emax_n = nx;
            emax_d = sx;
        }
    }
    double err = h * (emax_n / emax_d);

#pragma unroll
    for (int k = 0; k < 3; ++k) {
        R.xi[k] = xs[k];
        R.xa[k] = xs[3 + k];
        R.vi[k] = vn[k];
        R.va[k] = vn[3 + k];
        R.Ai[k] = A[6][k];
        R.Aa[k] = A[6][3 + k];
    }
    // observables at the step end: d = x_atom - x_ion, u = v_atom - v_ion
    const double u0 = vn[3] - vn[0], u1 = vn[4] - vn[1], u2 = vn[5] - vn[2];
    const double e0 = xs[3] - xs[0], e1 = xs[4] - xs[1], e2 = xs[5] - xs[2];
    const double s = fma(e2, u2, fma(e1, u1, e0 * u0));
    // a non-finite state or force makes the estimate NaN (it must reject, like the oracle's NaN)
    const bool finite_ok = (r2 > 0.0) && (r2 < 1.0e300) && (fabs(s) < 1.0e300);
    if (!finite_ok) err = __longlong_as_double(0x7ff8000000000000LL);
    R.t_new = t_new;
    R.err = err;
    R.r2 = r2;
    R.s = s;
}

// O3.3: clamp the step, detect the last step; called at t0 and after every accepted step.
__device__ __forceinline__ void prepare_step(const KParams& P, Traj& T)
{
    const double hmin = hmin_of(T.t);
    double h = fmin(P.hmax, fmax(hmin, T.h));
    const double rem = P.t_max - T.t;
    T.last = false;
    if (1.1 * h >= rem) {
        h = rem;
        T.last = true;
    }
    T.h = h;
    T.nofailed = true;
}

// Load-time initialisation (O3.1-O3.2 + observables at t0).  y = y0 of this trajectory.
template <int TRAP>
__device__ __forceinline__ void init_traj(const KParams& P, Traj& T)
{
    T.t = P.t0;
    double cs = 1.0;
    if (TRAP == TRAP_RF) cs = cos(P.omega * P.t0);
    double r2;
    accel<TRAP>(P, cs, T.xi, T.xa, T.Ai, T.Aa, r2);
    const double u0 = T.va[0] - T.vi[0], u1 = T.va[1] - T.vi[1], u2 = T.va[2] - T.vi[2];
    const double e0 = T.xa[0] - T.xi[0], e1 = T.xa[1] - T.xi[1], e2 = T.xa[2] - T.xi[2];
    T.sprev = fma(e2, u2, fma(e1, u1, e0 * u0));
    T.rmin2 = r2;
    T.t_first = 0.0;
    T.t_last = 0.0;
    T.n_acc = T.n_rej = T.n_turn = 0;
    T.any_min = false;
    // initial step: rho = max_i |f_i| / max(|y_i|, thr) / (0.8 rtol^(1/5))
    double rho = 0.0;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        rho = fmax(rho, fabs(T.vi[k]) / fmax(fabs(T.xi[k]), P.thr));
        rho = fmax(rho, fabs(T.Ai[k]) / fmax(fabs(T.vi[k]), P.thr));
        rho = fmax(rho, fabs(T.va[k]) / fmax(fabs(T.xa[k]), P.thr));
        rho = fmax(rho, fabs(T.Aa[k]) / fmax(fabs(T.va[k]), P.thr));
    }
    rho *= P.rho_scale;
    double h = fmin(P.hmax, P.t_max - P.t0);
    if (h * rho > 1.0) h = 1.0 / rho;
    T.h = fmax(h, hmin_of(T.t));
    prepare_step(P, T);
}

// Accept / reject logic of one attempt (O3.5-O3.8).  Returns the stop status (>= 0) when the
// trajectory has ended, -1 otherwise.  On return T holds the state to continue from (or the
// final state).
__device__ __forceinline__ int finish_attempt(const KParams& P, Traj& T, const Attempt& R)
{
    const double err = R.err;
    const double z = inv_fifth_root(err * P.inv_rtol);  // (err/rtol)^(-1/5)
    if (!(err <= P.rtol)) {
        // failed attempt
        T.n_rej++;
        const double hmin = hmin_of(T.t);
        if (T.h <= hmin) return 3;
        double fac = 0.5;
        if (T.nofailed) {
            fac = (err == err) ? fmax(0.1, 0.8 * z) : 0.1;
            T.nofailed = false;
        }
        T.h = fmax(hmin, T.h * fac);
        T.last = false;
        return -1;
    }
    // accepted
    T.n_acc++;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        T.xi[k] = R.xi[k];
        T.vi[k] = R.vi[k];
        T.xa[k] = R.xa[k];
        T.va[k] = R.va[k];
        T.Ai[k] = R.Ai[k];
        T.Aa[k] = R.Aa[k];
    }
    T.t = R.t_new;
    T.rmin2 = fmin(T.rmin2, R.r2);
    if (T.sprev < 0.0 && R.s >= 0.0) {  // radial minimum
        T.any_min = true;
        if (R.r2 < P.r_turn2) {
            T.n_turn++;
            if (T.n_turn == 1) T.t_first = R.t_new;
            T.t_last = R.t_new;
        }
    }
    T.sprev = R.s;
    if (T.any_min && R.r2 > P.r_exit2) return 0;
    if (T.last) return 1;
    if ((long long)T.n_acc >= P.max_steps) return 2;
    if (T.nofailed) T.h = (z < 6.25) ? T.h * (0.8 * z) : 5.0 * T.h;
    prepare_step(P, T);
    return -1;
}

// angle in [0, pi] between two 3-vectors: atan2(|u x v|, u.v)
__device__ __forceinline__ double angle_between(const double (&u)[3], const double (&v)[3])
{
    const double cx = u[1] * v[2] - u[2] * v[1];
    const double cy = u[2] * v[0] - u[0] * v[2];
    const double cz = u[0] * v[1] - u[1] * v[0];
    const double dot = fma(u[2], v[2], fma(u[1], v[1], u[0] * v[0]));
    return atan2(sqrt(fma(cz, cz, fma(cy, cy, cx * cx))), dot);
}

}  // namespace aig
