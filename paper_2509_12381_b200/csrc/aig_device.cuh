// aig_device.cuh -- device-side Dormand-Prince 5(4) stepper for the atom-ion ODE (sm_100a).
//
// What it computes: PAPER.md:71-90 (eq. (3)-(10)) integrated with the ode45 algorithm
// (constants: DESIGN.md "Integration loop").  How it computes it is
// B200-first and differs from the paper's seven pasted copies of f:
//   * the force depends on positions and time only, so the seven stages carry the six
//     ACCELERATION components only (Nystrom form, see gen_nystrom_tableau.py) -- 42 stage
//     doubles instead of 84, which is what lets a whole trajectory live in registers;
//   * in that form the position of stage s needs the accelerations of stages <= s-2 only, so
//     the six new force evaluations of a step form THREE dependent levels of two independent
//     evaluations each (stages 2|3, 4|5, 6|7).  The step is written level by level and is
//     branch-free (own reciprocal and cos), so the scheduler interleaves the two chains of a
//     level: FP64 latency is 8 cycles at 2 cycles issue per warp on sm_100a, a lone dependent
//     chain leaves 3/4 of the pipe idle;
//   * (dV/dr)/r = 4 C4/r^6 - 8 C8/r^10 needs even powers of r only: no square root;
//     1/r^2 = MUFU.RCP64H seed + one cubic and one Newton correction (no slow-path branch);
//   * cos(Omega t): Cody-Waite reduction + Taylor kernel (trig_constants.inc), five per attempt
//     (c6 = c7 = 1 share one, k1 is FSAL), all issued up front;
//   * the error norm is a maximum of ratios found by cross-multiplication in a fixed binary
//     tree and divided once; the controller's fifth root is a float seed + one cubic correction.
// Every product-sum is an explicit fma() and the library is compiled with -fmad=false, so the
// arithmetic of a trajectory does not depend on which kernel executes it: the per-thread
// integrator below and the six-lanes-per-trajectory one (aig_split.cuh) call the same scalar
// functions, and every sum that the split kernel forms across lanes (|d|^2, d.u, the error-norm
// tree) is written here with the same operands in the same order.  Results are therefore
// bit-identical whatever the schedule decides (tests/test_gpu_parity.py::test_schedule_invariance).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace aig {

#include "dp45_nystrom_tableau.inc"
#include "trig_constants.inc"

// TRAP_RF_BIG: RF trap with |Omega t| >= kCosMaxArg somewhere in the time span: libdevice cos
// (Payne-Hanek slow path available); chosen on the host, never needed by BASELINE.json's configs.
enum TrapMode { TRAP_NONE = 0, TRAP_STATIC = 1, TRAP_RF = 2, TRAP_RF_BIG = 3 };

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

// 1/x for normal x > 0: MUFU.RCP64H seed (20 bits), cubic correction y(1 + e + e^2), one Newton
// step.  Agrees with the IEEE quotient 1.0/x on every sampled input (measured on B200); no range
// check: x = 0, inf or NaN give NaN or 0, which the caller's finiteness test turns into a reject.
__device__ __forceinline__ double rcp_nr(double x)
{
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double e = fma(-x, y, 1.0);
    const double t = fma(e, e, e);
    y = fma(y, t, y);
    const double e1 = fma(-x, y, 1.0);
    return fma(y, e1, y);
}

// cos(x) for |x| < kCosMaxArg, branch-free (gen_trig_constants.py): k = round(x 2/pi),
// r = x - k pi/2 in three FMA steps, then the cos or sin Taylor kernel in z = r^2 chosen by k mod 2
// (coefficient table indexed, no select chain) and the sign by (k+1) mod 4 >= 2.
__device__ __forceinline__ double cos_cw(double x)
{
    const double kd = fma(x, kTwoOverPi, kRoundMagic);
    const int q = __double2loint(kd);
    const double k = kd - kRoundMagic;
    double r = fma(-k, kPio2_1, x);
    r = fma(-k, kPio2_2, r);
    r = fma(-k, kPio2_3, r);
    const int odd = q & 1;
    const double z = r * r;
    double p = kTrig[odd][kTrigTerms - 1];
#pragma unroll
    for (int i = kTrigTerms - 2; i >= 0; --i) p = fma(p, z, kTrig[odd][i]);
    const double base = odd ? r : 1.0;
    const double res = fma(base * z, p, base);
    return ((q + 1) & 2) ? -res : res;
}

template <int TRAP>
__device__ __forceinline__ double trap_cos(const KParams& P, double t)
{
    if (TRAP == TRAP_RF) return cos_cw(P.omega * t);
    if (TRAP == TRAP_RF_BIG) return cos(P.omega * t);
    return 1.0;
}

// (a + b) + c: the one order in which every three-component sum is formed (both kernels)
__device__ __forceinline__ double sum3(double a, double b, double c) { return (a + b) + c; }

// -(dV/dr)/(r m_ion) and +(dV/dr)/(r m_atom) from r^2:  (dV/dr)/r = 4 C4/r^6 - 8 C8/r^10
__device__ __forceinline__ void force_factors(const KParams& P, double r2, double& gi, double& ga)
{
    const double inv2 = rcp_nr(r2);
    const double inv4 = inv2 * inv2;
    const double inv6 = inv4 * inv2;
    const double g = inv6 * fma(-P.c8x8, inv4, P.c4x4);
    ga = g * P.inv_ma;
    gi = -(g * P.inv_mi);
}

// trap stiffness of one axis at cos(Omega t) = cs: w = wa + wb cs
template <int TRAP>
__device__ __forceinline__ double trap_w(double wa, double wb, double cs)
{
    return (TRAP == TRAP_STATIC) ? wa : fma(wb, cs, wa);
}

// Accelerations of both particles at positions (xi, xa), cos(Omega t) = cs.
// eq. (4)-(6): ion  acc_k = -(1/m_i)(dV/dr)(d_k/r) - w_k(t) x_k ;  eq. (8)-(10): atom acc_k = +(1/m_a)(dV/dr)(d_k/r)
// with d = x_ion - x_atom.  X = (xi, xa), Aout = (Ai, Aa).
template <int TRAP>
__device__ __forceinline__ void accel(const KParams& P, double cs, const double (&X)[6], double (&Aout)[6],
                                      double& r2_out)
{
    const double d0 = X[0] - X[3], d1 = X[1] - X[4], d2 = X[2] - X[5];
    const double r2 = sum3(d0 * d0, d1 * d1, d2 * d2);
    double gi, ga;
    force_factors(P, r2, gi, ga);
    Aout[3] = ga * d0;
    Aout[4] = ga * d1;
    Aout[5] = ga * d2;
    if (TRAP == TRAP_NONE) {
        Aout[0] = gi * d0;
        Aout[1] = gi * d1;
        Aout[2] = gi * d2;
    } else {
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const double w = trap_w<TRAP>(P.wa[k], P.wb[k], cs);
            const double dk = (k == 0) ? d0 : (k == 1 ? d1 : d2);
            Aout[k] = fma(-w, X[k], gi * dk);
        }
    }
    r2_out = r2;
}

// Position component of stage S+1 (S = 1..6): x + c h v + h^2 sum_{l <= S-2} abar_{S,l} A_l
// (older stages first, so the newest acceleration closes the chain).  A[l] = this component's A_l.
template <int S>
__device__ __forceinline__ double stage_pos(double x, double v, double hc, double h2, const double (&A)[7])
{
    const double base = fma(hc, v, x);
    if (S < 2) return base;
    double acc = kAbar[S][0] * A[0];
#pragma unroll
    for (int l = 1; l <= S - 2; ++l) {
        if (S == 6 && l == 1) continue;  // abar_72 = 0 exactly
        acc = fma(kAbar[S][l], A[l], acc);
    }
    return fma(h2, acc, base);
}

// 16 * (spacing of doubles above |t|): ode45's hmin = 16 eps(t)
__device__ __forceinline__ double hmin_of(double t)
{
    const double at = fabs(t);
    const double up = __longlong_as_double(__double_as_longlong(at) + 1LL);
    return 16.0 * (up - at);
}

// q^(-1/5) for q > 0: float seed (MUFU lg2/ex2, ~1e-7) + one cubic correction
// z (1 + rho/5 + 3 rho^2/25), rho = 1 - q z^5 (Taylor of (1-rho)^(-1/5)); relative error ~1e-16.
// q is clamped to [1e-30, 1e30] (the result is clamped by the caller).
__device__ __forceinline__ double inv_fifth_root(double q)
{
    q = fmin(fmax(q, 1e-30), 1e30);
    const double z = (double)exp2f(-0.2f * __log2f((float)q));
    const double z2 = z * z;
    const double z4 = z2 * z2;
    const double rho = fma(-q, z4 * z, 1.0);
    const double t = rho * fma(0.12, rho, 0.2);
    return fma(z, t, z);
}

// A candidate of the error norm: the ratio n/d with d > 0, kept unevaluated.
struct Ratio {
    double n, d;
};
// the larger of two ratios by cross-multiplication (all denominators > 0); ties keep a
__device__ __forceinline__ Ratio ratio_max(const Ratio a, const Ratio b)
{
    const bool gt = b.n * a.d > a.n * b.d;
    Ratio r;
    r.n = gt ? b.n : a.n;
    r.d = gt ? b.d : a.d;
    return r;
}

// Step end of component i (velocity and both error rows), from its seven stage accelerations:
//   v_new = v + h sum b_l A_l ; e_v = sum E_l A_l ; e_x = h sum Ebar_l A_l  (b_2 = E_2 = Ebar_2 = b_7 = Ebar_7 = 0)
// returns v_new and the two norm candidates |e_v| / max(|v|,|v_new|,thr), |e_x| / max(|x|,|x_new|,thr).
__device__ __forceinline__ double step_end_component(const KParams& P, double h, double x, double xn, double v,
                                                     const double (&A)[7], Ratio& cv, Ratio& cx)
{
    double sb = kB[0] * A[0];
    sb = fma(kB[2], A[2], sb);
    sb = fma(kB[3], A[3], sb);
    sb = fma(kB[4], A[4], sb);
    sb = fma(kB[5], A[5], sb);
    const double vn = fma(h, sb, v);
    double ev = kE[0] * A[0];
    ev = fma(kE[2], A[2], ev);
    ev = fma(kE[3], A[3], ev);
    ev = fma(kE[4], A[4], ev);
    ev = fma(kE[5], A[5], ev);
    ev = fma(kE[6], A[6], ev);
    double ex = kEbar[0] * A[0];
    ex = fma(kEbar[2], A[2], ex);
    ex = fma(kEbar[3], A[3], ex);
    ex = fma(kEbar[4], A[4], ex);
    ex = fma(kEbar[5], A[5], ex);
    ex = ex * h;
    cv.n = fabs(ev);
    cv.d = fmax(fmax(fabs(v), fabs(vn)), P.thr);
    cx.n = fabs(ex);
    cx.d = fmax(fmax(fabs(x), fabs(xn)), P.thr);
    return vn;
}

// max over the six candidates of one particle (fixed tree: ((v0,x0),(v1,x1)) , (v2,x2))
__device__ __forceinline__ Ratio particle_norm(const Ratio (&cv)[3], const Ratio (&cx)[3])
{
    const Ratio a = ratio_max(cv[0], cx[0]);
    const Ratio b = ratio_max(cv[1], cx[1]);
    const Ratio c = ratio_max(cv[2], cx[2]);
    return ratio_max(ratio_max(a, b), c);
}

// Controller state of one trajectory: time, step size, radial observable at t, accepted-step
// count and flags.  The split kernel keeps a copy on each of a trajectory's six lanes.
struct Core {
    double t, h, sprev;
    int n_acc;
    unsigned flags;  // kAnyMin | kLast | kNoFailed (one register instead of three)
};
constexpr unsigned kAnyMin = 1u;    // a radial minimum has been seen (arms the exit test)
constexpr unsigned kLast = 2u;      // this attempt ends exactly at t_max
constexpr unsigned kNoFailed = 4u;  // no failed attempt since the last accepted step

// Per-lane state of one trajectory in the per-thread integrator (registers).  X = (x_ion, x_atom),
// V likewise, A1 = the accelerations at (t, y): stage 1, FSAL.
struct Traj {
    double X[6], V[6], A1[6];
    Core c;
};

// The rarely touched part of a trajectory's state (observables and counters).  The per-thread
// integrator keeps it in shared memory (ColdShared in aig_kernels.cu: one slot per thread, SoA)
// to stay within 168 registers at three blocks per SM; ColdRegs is the same thing in registers.
struct ColdRegs {
    double rmin2_, t_first_, t_last_;
    int n_rej_, n_turn_;
    __device__ __forceinline__ double& rmin2() { return rmin2_; }
    __device__ __forceinline__ double& t_first() { return t_first_; }
    __device__ __forceinline__ double& t_last() { return t_last_; }
    __device__ __forceinline__ int& n_rej() { return n_rej_; }
    __device__ __forceinline__ int& n_turn() { return n_turn_; }
};

// Result of one attempted step (before accept / reject).
struct Attempt {
    double X[6], V[6], A7[6];  // ynew and f(t_new, ynew) accelerations (stage 7)
    double t_new, err, r2, s;  // r2, s: |d|^2 and d.u at ynew (observables)
};

// scaled error estimate from the two particle norms, NaN when the new state is not finite
__device__ __forceinline__ double error_estimate(double h, const Ratio ion, const Ratio atom, double r2, double s)
{
    const Ratio m = ratio_max(ion, atom);
    double err = h * (m.n * rcp_nr(m.d));
    // a non-finite state or force makes the estimate NaN (it must reject, like the oracle's NaN)
    const bool finite_ok = (r2 > 0.0) && (r2 < 1.0e300) && (fabs(s) < 1.0e300);
    if (!finite_ok) err = __longlong_as_double(0x7ff8000000000000LL);
    return err;
}

// radial observable s = (x_atom - x_ion).(v_atom - v_ion)
__device__ __forceinline__ double radial_s(const double (&X)[6], const double (&V)[6])
{
    const double u0 = V[3] - V[0], u1 = V[4] - V[1], u2 = V[5] - V[2];
    const double e0 = X[3] - X[0], e1 = X[4] - X[1], e2 = X[5] - X[2];
    return sum3(e0 * u0, e1 * u1, e2 * u2);
}

// One attempted Dormand-Prince step of size T.c.h from (T.c.t, y), stage 1 taken from T.A1.
template <int TRAP>
__device__ __forceinline__ void dp45_attempt(const KParams& P, const Traj& T, Attempt& R)
{
    const double h = T.c.h;
    const double h2 = h * h;
    const double t_new = (T.c.flags & kLast) ? P.t_max : T.c.t + h;

    // A[i][l]: acceleration component i (0-2 ion, 3-5 atom) of stage l+1
    double A[6][7];
#pragma unroll
    for (int i = 0; i < 6; ++i) A[i][0] = T.A1[i];
    double Xs[2][6], r2[2];
    // three levels; the two stages of a level are independent of each other
#pragma unroll
    for (int lev = 0; lev < 3; ++lev) {
        // cos(Omega t) at the stage times of this level (independent of the positions; c6 = c7 = 1)
        double cs[2];
        cs[0] = trap_cos<TRAP>(P, (lev == 2) ? t_new : fma(kC[2 * lev + 1], h, T.c.t));
        cs[1] = (lev == 2) ? cs[0] : trap_cos<TRAP>(P, fma(kC[2 * lev + 2], h, T.c.t));
#pragma unroll
        for (int e = 0; e < 2; ++e) {
            const int s = 2 * lev + 1 + e;  // stage s+1
            const double hc = h * kC[s];
#pragma unroll
            for (int i = 0; i < 6; ++i) {
                Xs[e][i] = (s == 1)   ? stage_pos<1>(T.X[i], T.V[i], hc, h2, A[i])
                           : (s == 2) ? stage_pos<2>(T.X[i], T.V[i], hc, h2, A[i])
                           : (s == 3) ? stage_pos<3>(T.X[i], T.V[i], hc, h2, A[i])
                           : (s == 4) ? stage_pos<4>(T.X[i], T.V[i], hc, h2, A[i])
                           : (s == 5) ? stage_pos<5>(T.X[i], T.V[i], hc, h2, A[i])
                                      : stage_pos<6>(T.X[i], T.V[i], hc, h2, A[i]);
            }
        }
#pragma unroll
        for (int e = 0; e < 2; ++e) {
            const int s = 2 * lev + 1 + e;
            double a[6];
            accel<TRAP>(P, cs[e], Xs[e], a, r2[e]);
#pragma unroll
            for (int i = 0; i < 6; ++i) A[i][s] = a[i];
        }
    }
    // Xs[1] = x_new (stage 7 position = 5th-order solution), A[.][6] = f(t_new, ynew)
    Ratio cv[6], cx[6];
#pragma unroll
    for (int i = 0; i < 6; ++i) {
        R.X[i] = Xs[1][i];
        R.V[i] = step_end_component(P, h, T.X[i], Xs[1][i], T.V[i], A[i], cv[i], cx[i]);
        R.A7[i] = A[i][6];
    }
    const Ratio cvi[3] = {cv[0], cv[1], cv[2]}, cxi[3] = {cx[0], cx[1], cx[2]};
    const Ratio cva[3] = {cv[3], cv[4], cv[5]}, cxa[3] = {cx[3], cx[4], cx[5]};
    R.s = radial_s(R.X, R.V);
    R.r2 = r2[1];
    R.t_new = t_new;
    R.err = error_estimate(h, particle_norm(cvi, cxi), particle_norm(cva, cxa), R.r2, R.s);
}

// O3.3: clamp the step, detect the last step; called at t0 and after every accepted step.
__device__ __forceinline__ void prepare_step(const KParams& P, Core& K)
{
    const double hmin = hmin_of(K.t);
    double h = fmin(P.hmax, fmax(hmin, K.h));
    const double rem = P.t_max - K.t;
    unsigned f = (K.flags & kAnyMin) | kNoFailed;
    if (1.1 * h >= rem) {
        h = rem;
        f |= kLast;
    }
    K.h = h;
    K.flags = f;
}

// Load-time initialisation (O3.1-O3.2 + observables at t0).  T.X, T.V = y0 of this trajectory.
template <int TRAP, class Cold>
__device__ __forceinline__ void init_traj(const KParams& P, Traj& T, Cold& C)
{
    Core& K = T.c;
    K.t = P.t0;
    const double cs = trap_cos<TRAP>(P, P.t0);
    double r2;
    accel<TRAP>(P, cs, T.X, T.A1, r2);
    K.sprev = radial_s(T.X, T.V);
    C.rmin2() = r2;
    C.t_first() = 0.0;
    C.t_last() = 0.0;
    K.n_acc = 0;
    C.n_rej() = 0;
    C.n_turn() = 0;
    K.flags = 0u;
    // initial step: rho = max_i |f_i| / max(|y_i|, thr) / (0.8 rtol^(1/5))
    double rho = 0.0;
#pragma unroll
    for (int i = 0; i < 6; ++i) {
        rho = fmax(rho, fabs(T.V[i]) / fmax(fabs(T.X[i]), P.thr));
        rho = fmax(rho, fabs(T.A1[i]) / fmax(fabs(T.V[i]), P.thr));
    }
    rho *= P.rho_scale;
    double h = fmin(P.hmax, P.t_max - P.t0);
    if (h * rho > 1.0) h = 1.0 / rho;
    K.h = fmax(h, hmin_of(K.t));
    prepare_step(P, K);
}

// Accept / reject logic of one attempt (O3.5-O3.8) on the controller state: err = the scaled
// error estimate, (t_new, r2, s) = time, |d|^2 and d.u at the attempted step end.  Sets
// `accepted`; returns the stop status (>= 0) when the trajectory has ended, -1 otherwise.  The
// caller moves ynew into y when `accepted` (also when the trajectory ends on this step).
template <class Cold>
__device__ __forceinline__ int finish_core(const KParams& P, Core& K, Cold& C, double err, double t_new,
                                           double r2, double s, bool& accepted)
{
    const double z = inv_fifth_root(err * P.inv_rtol);  // (err/rtol)^(-1/5)
    accepted = (err <= P.rtol);
    if (!accepted) {
        // failed attempt
        C.n_rej()++;
        const double hmin = hmin_of(K.t);
        if (K.h <= hmin) return 3;
        double fac = 0.5;
        if (K.flags & kNoFailed) fac = (err == err) ? fmax(0.1, 0.8 * z) : 0.1;
        K.h = fmax(hmin, K.h * fac);
        K.flags &= kAnyMin;  // clears kNoFailed and kLast
        return -1;
    }
    K.n_acc++;
    K.t = t_new;
    if (r2 < C.rmin2()) C.rmin2() = r2;
    if (K.sprev < 0.0 && s >= 0.0) {  // radial minimum
        K.flags |= kAnyMin;
        if (r2 < P.r_turn2) {
            const int nt = ++C.n_turn();
            if (nt == 1) C.t_first() = t_new;
            C.t_last() = t_new;
        }
    }
    K.sprev = s;
    if ((K.flags & kAnyMin) && r2 > P.r_exit2) return 0;
    if (K.flags & kLast) return 1;
    if ((long long)K.n_acc >= P.max_steps) return 2;
    if (K.flags & kNoFailed) K.h = (z < 6.25) ? K.h * (0.8 * z) : 5.0 * K.h;
    prepare_step(P, K);
    return -1;
}

// finish_core for the per-thread integrator: on return T holds the state to continue from (or
// the final state).
template <class Cold>
__device__ __forceinline__ int finish_attempt(const KParams& P, Traj& T, Cold& C, const Attempt& R)
{
    bool accepted;
    const int st = finish_core(P, T.c, C, R.err, R.t_new, R.r2, R.s, accepted);
    if (accepted) {
#pragma unroll
        for (int i = 0; i < 6; ++i) {
            T.X[i] = R.X[i];
            T.V[i] = R.V[i];
            T.A1[i] = R.A7[i];
        }
    }
    return st;
}

// angle in [0, pi] between two 3-vectors: atan2(|u x v|, u.v)
__device__ __forceinline__ double angle_between(const double (&u)[3], const double (&v)[3])
{
    const double cx = fma(u[1], v[2], -(u[2] * v[1]));
    const double cy = fma(u[2], v[0], -(u[0] * v[2]));
    const double cz = fma(u[0], v[1], -(u[1] * v[0]));
    const double dot = fma(u[2], v[2], fma(u[1], v[1], u[0] * v[0]));
    return atan2(sqrt(fma(cz, cz, fma(cy, cy, cx * cx))), dot);
}

}  // namespace aig
