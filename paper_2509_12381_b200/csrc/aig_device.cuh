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
//   * the relative position d = x_ion - x_atom has a stage chain of its own (the r^-9 wall would see
//     the rounding of a difference of two lab-frame positions): "Stage positions" below;
//   * (dV/dr)/r = 4 C4/r^6 - 8 C8/r^10 needs even powers of r only: no square root;
//     1/r^2 = MUFU.RCP64H seed + one cubic correction (three FMAs, no slow-path branch);
//   * cos(Omega t): Cody-Waite reduction + Taylor kernel (trig_constants.inc), five per attempt
//     (c6 = c7 = 1 share one, k1 is FSAL), all issued up front;
//   * the error norm is a maximum of ratios found by cross-multiplication in a fixed binary
//     tree and divided once; the controller's fifth root is a float seed + one Newton-type correction
//     folded into the new step size (grow_step).
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
// The kernels' template argument `TRAP` is a MODE: trap mode + 4 x potential kind.
//   potential kind 0: the benchmark potential V = C8/r^8 - C4/r^4, even powers of r only;
//   potential kind 1: V = C_m/r^m - C_n/r^n with integer exponents (NEXT-1).
enum PotKind { POT_4_8 = 0, POT_GENERAL = 1 };
__host__ __device__ constexpr int trap_of(int mode) { return mode & 3; }
__host__ __device__ constexpr int pot_of(int mode) { return mode >> 2; }

// Derived constants of one call; passed by value as a kernel argument (constant bank).
struct KParams {
    double g4i, g8i;        // -4 C4/m_ion, +8 C8/m_ion :  -(dV/dr)/(r m_ion)  = (g4i + g8i/r^4)/r^6
    double g4a, g8a;        // +4 C4/m_atom, -8 C8/m_atom : +(dV/dr)/(r m_atom) = (g4a + g8a/r^4)/r^6
                            // general potential: g4 = -/+ n C_n/m, g8 = +/- m C_m/m
    int pot_e_att, pot_e_rep;  // general potential: (dV/dr)/r = n C_n b^e_att - m C_m b^e_rep with b = 1/r^2
    int pot_sqrt;              //   (exponents (n+2)/2, (m+2)/2), or b = 1/r (exponents n+2, m+2) if n or m is odd
    double wa[3], wb[3];    // w_k(t) = wa_k + wb_k cos(Omega t): wa = a_k Om^2/4, wb = q_k Om^2/2
    double omega, half_omega;
    double t0, t_max, hmax; // hmax = 0.1 (t_max - t0)
    double rtol, inv_rtol, thr;  // thr = atol/rtol
    double rho_scale;       // 1/(0.8 rtol^(1/5)) for the initial step
    double r_exit2, r_turn2;     // squared radii; r_exit2 = +inf disables the exit stop
    long long max_steps;
};

// 1/x for normal x > 0: MUFU.RCP64H seed (relative error < 1e-6, measured) + one cubic correction
// y(1 + e + e^2), e = 1 - x y: error e^3 < 1e-18 plus one rounding.  Differs from the IEEE quotient
// 1.0/x by 1 ulp on 0.03 % of inputs and never by more (1e9 samples on B200); three dependent FMAs
// after the seed instead of libdevice's division.  No range check: x = 0, inf or NaN give NaN or 0,
// which the caller's finiteness test turns into a reject.
__device__ __forceinline__ double rcp_nr(double x)
{
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double e = fma(-x, y, 1.0);
    const double t = fma(e, e, e);
    return fma(y, t, y);
}

// cos(2 y) for |y| < kCosMaxArg, branch-free and table-free (gen_trig_constants.py): k = round(y 2/pi),
// u = y - k pi/2 in two FMA steps (|u| <= pi/4), s = sin u by its Taylor kernel in z = u^2 (two
// interleaved Horner chains in z^2: half the dependent depth), cos(2y) = (-1)^k (1 - 2 s^2).
// Absolute error < 2e-16 (the force only needs cos to absolute accuracy: it multiplies q_k).
__device__ __forceinline__ double cos2_cw(double y)
{
    const double kd = fma(y, kTwoOverPi, kRoundMagic);
    const int q = __double2loint(kd);
    const double k = kd - kRoundMagic;
    // two constants: the third one would change u by |k| 1.5e-33 < 1e-28 for |y| < kCosMaxArg
    double u = fma(-k, kPio2_1, y);
    u = fma(-k, kPio2_2, u);
    const double z = u * u;
    const double w = z * z;
    double pe = fma(kSin[6], w, kSin[4]);
    double po = fma(kSin[7], w, kSin[5]);
    pe = fma(pe, w, kSin[2]);
    po = fma(po, w, kSin[3]);
    pe = fma(pe, w, kSin[0]);
    po = fma(po, w, kSin[1]);
    const double p = fma(po, z, pe);
    const double sn = fma(u * z, p, u);
    const double res = fma(-2.0 * sn, sn, 1.0);
    return (q & 1) ? -res : res;
}

template <int TRAP>
__device__ __forceinline__ double trap_cos(const KParams& P, double t)
{
    if (trap_of(TRAP) == TRAP_RF) return cos2_cw(P.half_omega * t);
    if (trap_of(TRAP) == TRAP_RF_BIG) return cos(P.omega * t);
    return 1.0;
}

// (a + b) + c: the one order in which every three-component sum is formed (both kernels)
__device__ __forceinline__ double sum3(double a, double b, double c) { return (a + b) + c; }

// plain compare-and-select maximum / minimum: one DSETP and two selects.  Written in PTX because
// the compiler turns (a > b) ? a : b into max.f64, whose SASS expansion (DSETP.MAX, FSEL, SEL, a
// predicated LOP3 that quiets NaNs) is longer and deeper; the callers do not need NaN quieting.
// A NaN first operand yields the second operand.
__device__ __forceinline__ double dmax(double a, double b)
{
    double r;
    asm("{\n\t.reg .pred p;\n\tsetp.gt.f64 p, %1, %2;\n\tselp.f64 %0, %1, %2, p;\n\t}" : "=d"(r) : "d"(a), "d"(b));
    return r;
}
__device__ __forceinline__ double dmin(double a, double b)
{
    double r;
    asm("{\n\t.reg .pred p;\n\tsetp.lt.f64 p, %1, %2;\n\tselp.f64 %0, %1, %2, p;\n\t}" : "=d"(r) : "d"(a), "d"(b));
    return r;
}

// gi = -(dV/dr)/(r m_ion) and ga = +(dV/dr)/(r m_atom) from r^2, (dV/dr)/r = 4 C4/r^6 - 8 C8/r^10:
// the masses are folded into the constants so that both factors are three operations behind 1/r^2
// x^e for an integer e >= 1 by repeated squaring; the order of the products is fixed by e alone
__device__ __forceinline__ double ipow(double x, int e)
{
    double r = 1.0, b = x;
    for (;;) {
        if (e & 1) r *= b;
        e >>= 1;
        if (e == 0) break;
        b *= b;
    }
    return r;
}
template <int MODE>
__device__ __forceinline__ void force_factors(const KParams& P, double r2, double& gi, double& ga)
{
    const double inv2 = rcp_nr(r2);
    if (pot_of(MODE) == POT_4_8) {
        const double inv4 = inv2 * inv2;
        const double inv6 = inv4 * inv2;
        gi = inv6 * fma(P.g8i, inv4, P.g4i);
        ga = inv6 * fma(P.g8a, inv4, P.g4a);
    } else {
        // V = C_m/r^m - C_n/r^n: (dV/dr)/r = n C_n/r^(n+2) - m C_m/r^(m+2), powers of 1/r^2 (or of 1/r
        // when an exponent is odd: one square root)
        const double b = P.pot_sqrt ? sqrt(inv2) : inv2;
        const double pa = ipow(b, P.pot_e_att), pr = ipow(b, P.pot_e_rep);
        gi = fma(P.g8i, pr, P.g4i * pa);
        ga = fma(P.g8a, pr, P.g4a * pa);
    }
}

// trap stiffness of one axis at cos(Omega t) = cs: w = wa + wb cs
template <int TRAP>
__device__ __forceinline__ double trap_w(double wa, double wb, double cs)
{
    return (trap_of(TRAP) == TRAP_STATIC) ? wa : fma(wb, cs, wa);
}

// Accelerations of both particles from the relative position D = x_ion - x_atom and the ion position
// Xi (the trap acts on the ion only), cos(Omega t) = cs.
// eq. (4)-(6): ion  acc_k = -(1/m_i)(dV/dr)(d_k/r) - w_k(t) x_k  [the trap product first: it does not wait for 1/r^2];  eq. (8)-(10): atom acc_k = +(1/m_a)(dV/dr)(d_k/r).
// Aout = (Ai, Aa).
template <int TRAP>
__device__ __forceinline__ void accel(const KParams& P, double cs, const double (&D)[3], const double (&Xi)[3],
                                      double (&Aout)[6], double& r2_out)
{
    const double d0 = D[0], d1 = D[1], d2 = D[2];
    const double r2 = sum3(d0 * d0, d1 * d1, d2 * d2);
    double gi, ga;
    force_factors<TRAP>(P, r2, gi, ga);
    Aout[3] = ga * d0;
    Aout[4] = ga * d1;
    Aout[5] = ga * d2;
    if (trap_of(TRAP) == TRAP_NONE) {
        Aout[0] = gi * d0;
        Aout[1] = gi * d1;
        Aout[2] = gi * d2;
    } else {
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const double w = trap_w<TRAP>(P.wa[k], P.wb[k], cs);
            const double dk = (k == 0) ? d0 : (k == 1 ? d1 : d2);
            Aout[k] = fma(gi, dk, -(w * Xi[k]));
        }
    }
    r2_out = r2;
}

// Stage positions (Nystrom form).  Stage S+1 (S = 1..6) sits at x + c h v + h^2 sum_{l <= S-2} abar_{S,l} A_l
// (older stages first, so the newest acceleration closes the chain); A[l] = this component's A_l.
// The force needs the RELATIVE position d = x_ion - x_atom, at the repulsive wall to far better than
// the spacing of doubles at |x| ~ 1e3 a0 (the force goes as r^-9 with r ~ 7.6 a0: a difference of two
// rounded lab-frame stage positions would carry eps |x| / r ~ 1e-14 into r and ten times that into the
// force).  So the relative position has a chain of its own, started from d(t) = x_ion - x_atom and
// u(t) = v_ion - v_atom at the beginning of the step:
//     d_s = d + c h u + h^2 (acc_ion - acc_atom),   acc = sum_l abar_{S,l} A_l,
// accurate to the spacing of doubles at |d|.  The ion's own stage position is still formed (the trap
// force needs it, to ordinary accuracy), the atom's only at the step end (stage 7 = the new state).
template <int S>
__device__ __forceinline__ double stage_acc(const double (&A)[7])
{
    static_assert(S >= 2 && S <= 6, "stages 3..7");
    double acc = kAbar[S][0] * A[0];
#pragma unroll
    for (int l = 1; l <= S - 2; ++l) {
        if (S == 6 && l == 1) continue;  // abar_72 = 0 exactly
        acc = fma(kAbar[S][l], A[l], acc);
    }
    return acc;
}
// x + c h v + h^2 acc  (also the relative position, with x -> d, v -> u, acc -> acc_ion - acc_atom)
__device__ __forceinline__ double stage_pos(double x, double v, double hc, double h2, double acc)
{
    return fma(h2, acc, fma(hc, v, x));
}

// 16 * (spacing of doubles above |t|): ode45's hmin = 16 eps(t)
__device__ __forceinline__ double hmin_of(double t)
{
    const double at = fabs(t);
    const double up = __longlong_as_double(__double_as_longlong(at) + 1LL);
    return 16.0 * (up - at);
}

// The controller's fifth root, q = err / rtol.  Float seed z ~ q^(-1/5) (MUFU lg2 / ex2, relative error
// ~1e-7) and one Newton-type correction z (1 + rho/5), rho = 1 - q z^5 (first term of the Taylor series of
// (1 - rho)^(-1/5); the next one, 3 rho^2/25, is ~1e-13: far below the rounding noise of the error estimate
// the step size is derived from).
__device__ __forceinline__ float fifth_root_seed(float qf)
{
    float lg, zf;
    asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(lg) : "f"(qf));
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(zf) : "f"(-0.2f * lg));
    return zf;
}
// q^(-1/5), q clamped to [1e-30, 1e30] (the reject path: the result is clamped by the caller)
__device__ __forceinline__ double inv_fifth_root(double q)
{
    // clamp the seed in float (two 4-cycle FMNMX instead of two FP64 compare/select pairs on the
    // controller's dependent chain); the operand and the result are normal floats after the clamp
    const double z = (double)fifth_root_seed(fminf(fmaxf((float)q, 1e-30f), 1e30f));
    q = dmin(dmax(q, 1e-30), 1e30);  // off the chain: only the correction needs it
    const double z2 = z * z;
    const double rho = fma(-(q * z), z2 * z2, 1.0);
    return fma(z, 0.2 * rho, z);
}
// Step size after an accepted step without failures (O3.7): 0.8 h (rtol/err)^(1/5), at most 5 h.  One
// expression for both kernels, arranged for a short dependent chain behind the seed:
//     rho = 1 - (q z) z^4,   h_grow = (0.8 h z)(1 + rho/5) = fma(0.8 h z, rho/5, 0.8 h z),   5 h if z >= 6.25
// (the growth limit is decided on the seed: at z = 6.25 the two branches agree to 1e-7 anyway).  q and its
// float image qf are taken as given: the caller clamps them to [1e-30, 1e30] or knows that q <= 1, where
// the clamps change nothing (q < 1e-30 or q = 0 end in 5 h either way: z >= 1e6, or NaN products).
__device__ __forceinline__ double grow_step(double h, double q, float qf)
{
    const float zf = fifth_root_seed(qf);
    const double z = (double)zf;
    const double z2 = z * z;
    const double qz = q * z;
    const double h08z = (0.8 * h) * z;
    const double rho = fma(-qz, z2 * z2, 1.0);
    const double hz = fma(h08z, 0.2 * rho, h08z);
    return (zf < 6.25f) ? hz : 5.0 * h;
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
// in two pieces so that everything that does not need stages 6 and 7 (the last level) can be issued
// while that level's force evaluation is in flight.
struct StepEndPart {
    double sb, ev, ex;  // the three sums over stages 1, 3, 4, 5
    double mv, mx;      // max(|v|, thr), max(|x|, thr)
};
__device__ __forceinline__ void step_end_begin(const KParams& P, double x, double v, const double (&A)[7],
                                               StepEndPart& S)
{
    double sb = kB[0] * A[0];
    sb = fma(kB[2], A[2], sb);
    sb = fma(kB[3], A[3], sb);
    S.sb = fma(kB[4], A[4], sb);
    double ev = kE[0] * A[0];
    ev = fma(kE[2], A[2], ev);
    ev = fma(kE[3], A[3], ev);
    S.ev = fma(kE[4], A[4], ev);
    double ex = kEbar[0] * A[0];
    ex = fma(kEbar[2], A[2], ex);
    ex = fma(kEbar[3], A[3], ex);
    S.ex = fma(kEbar[4], A[4], ex);
    S.mv = dmax(fabs(v), P.thr);
    S.mx = dmax(fabs(x), P.thr);
}

// returns v_new and the two norm candidates |e_v| / max(|v|,|v_new|,thr), |e_x| / max(|x|,|x_new|,thr)
__device__ __forceinline__ double step_end_finish(const StepEndPart& S, double h, double xn, double v, double A6,
                                                  double A7, Ratio& cv, Ratio& cx)
{
    const double vn = fma(h, fma(kB[5], A6, S.sb), v);
    const double ev = fma(kE[6], A7, fma(kE[5], A6, S.ev));
    const double ex = fma(kEbar[5], A6, S.ex) * h;
    cv.n = fabs(ev);
    cv.d = dmax(fabs(vn), S.mv);
    cx.n = fabs(ex);
    cx.d = dmax(fabs(xn), S.mx);
    return vn;
}

// Largest of the four ratios of one axis k (velocity and position rows of both particles), found by
// cross-multiplication in a fixed tree and divided once: max_i |e_i| / max(|y_i|, |ynew_i|, thr)
// over the four components of that axis.  The error norm is the maximum of the three axis values
// (an exact maximum: its order does not matter, so the split kernel can gather them in any order).
__device__ __forceinline__ double axis_quotient(const Ratio cvi, const Ratio cxi, const Ratio cva, const Ratio cxa)
{
    const Ratio m = ratio_max(ratio_max(cvi, cxi), ratio_max(cva, cxa));
    return m.n * rcp_nr(m.d);
}

// The same quotient with the four reciprocals taken BEFORE the maximum is known (the six-lane kernel: three more
// reciprocals issued, four fewer operations on the dependent chain).  The reciprocal travels with its ratio through
// the same cross-multiplication tree, so the result is m.n * rcp_nr(m.d) of the same m: the same bits.
struct RatioR {
    double n, d, r;
};
__device__ __forceinline__ RatioR ratio_max_r(const RatioR a, const RatioR b)
{
    const bool gt = b.n * a.d > a.n * b.d;
    RatioR m;
    m.n = gt ? b.n : a.n;
    m.d = gt ? b.d : a.d;
    m.r = gt ? b.r : a.r;
    return m;
}
__device__ __forceinline__ double axis_quotient_early_rcp(const Ratio cvi, const Ratio cxi, const Ratio cva, const Ratio cxa)
{
    const RatioR a{cvi.n, cvi.d, rcp_nr(cvi.d)}, b{cxi.n, cxi.d, rcp_nr(cxi.d)}, c{cva.n, cva.d, rcp_nr(cva.d)},
        d{cxa.n, cxa.d, rcp_nr(cxa.d)};
    const RatioR m = ratio_max_r(ratio_max_r(a, b), ratio_max_r(c, d));
    return m.n * m.r;
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
// integrator keeps it in shared memory (ColdShared in aig_kernels.cu: one slot per thread, SoA:
// that is what lets it run at 168 registers, three blocks of 128 threads per SM, without a spill);
// ColdRegs is the same thing in registers.
struct ColdRegs {
    static constexpr bool kInRegisters = true;
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

// scaled error estimate from the three axis quotients, NaN when the new state is not finite
// (in two pieces: the six-lane integrator tests the second one in its fast-path vote)
__device__ __forceinline__ double error_raw(double h, double q0, double q1, double q2)
{
    return h * dmax(dmax(q0, q1), q2);
}
__device__ __forceinline__ bool attempt_finite(double q0, double q1, double q2, double r2, double s)
{
    return (r2 > 0.0) & (r2 < 1.0e300) & (fabs(s) < 1.0e300) & (q0 == q0) & (q1 == q1) & (q2 == q2);
}
__device__ __forceinline__ double error_estimate(double h, double q0, double q1, double q2, double r2, double s)
{
    double err = error_raw(h, q0, q1, q2);
    // a non-finite state or force makes the estimate NaN (it must reject, like the oracle's NaN)
    if (!attempt_finite(q0, q1, q2, r2, s)) err = __longlong_as_double(0x7ff8000000000000LL);
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
    // relative position and velocity at the beginning of the step
    double d0[3], u0[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        d0[k] = T.X[k] - T.X[3 + k];
        u0[k] = T.V[k] - T.V[3 + k];
    }
    double Ds[2][3], Xis[2][3], Xa_new[3], r2[2];
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
            for (int k = 0; k < 3; ++k) {
                if (s == 1) {
                    Xis[e][k] = fma(hc, T.V[k], T.X[k]);
                    Ds[e][k] = fma(hc, u0[k], d0[k]);
                } else {
                    const double ai = (s == 2)   ? stage_acc<2>(A[k])
                                      : (s == 3) ? stage_acc<3>(A[k])
                                      : (s == 4) ? stage_acc<4>(A[k])
                                      : (s == 5) ? stage_acc<5>(A[k])
                                                 : stage_acc<6>(A[k]);
                    const double aa = (s == 2)   ? stage_acc<2>(A[3 + k])
                                      : (s == 3) ? stage_acc<3>(A[3 + k])
                                      : (s == 4) ? stage_acc<4>(A[3 + k])
                                      : (s == 5) ? stage_acc<5>(A[3 + k])
                                                 : stage_acc<6>(A[3 + k]);
                    Xis[e][k] = stage_pos(T.X[k], T.V[k], hc, h2, ai);
                    Ds[e][k] = stage_pos(d0[k], u0[k], hc, h2, ai - aa);
                    if (s == 6) Xa_new[k] = stage_pos(T.X[3 + k], T.V[3 + k], hc, h2, aa);
                }
            }
        }
#pragma unroll
        for (int e = 0; e < 2; ++e) {
            const int s = 2 * lev + 1 + e;
            double a[6];
            accel<TRAP>(P, cs[e], Ds[e], Xis[e], a, r2[e]);
#pragma unroll
            for (int i = 0; i < 6; ++i) A[i][s] = a[i];
        }
    }
    // stage 7 position = the 5th-order solution x_new; A[.][6] = f(t_new, ynew).  Axis by axis (ion and atom
    // component of the axis, then its quotient at once: eight norm candidates live instead of twenty-four)
    double q[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        Ratio cv[2], cx[2];
#pragma unroll
        for (int pa = 0; pa < 2; ++pa) {
            const int i = k + 3 * pa;
            R.X[i] = pa ? Xa_new[k] : Xis[1][k];
            StepEndPart S;
            step_end_begin(P, T.X[i], T.V[i], A[i], S);
            R.V[i] = step_end_finish(S, h, R.X[i], T.V[i], A[i][5], A[i][6], cv[pa], cx[pa]);
            R.A7[i] = A[i][6];
        }
        q[k] = axis_quotient(cv[0], cx[0], cv[1], cx[1]);
    }
    R.s = radial_s(R.X, R.V);
    R.r2 = r2[1];
    R.t_new = t_new;
    R.err = error_estimate(h, q[0], q[1], q[2], R.r2, R.s);
}

// Times of one attempt that depend on (t, h) only: the split kernel forms them while the stages
// are in flight, so that the controller's dependent chain after the error estimate is short.
struct StepTimes {
    double t_new;     // end of the attempted step (exactly t_max on the last one)
    double hmin_cur;  // hmin at t (reject path)
    double hmin_new;  // hmin at t_new
    double rem_new;   // t_max - t_new
};
__device__ __forceinline__ StepTimes step_times(const KParams& P, const Core& K)
{
    StepTimes S;
    S.t_new = (K.flags & kLast) ? P.t_max : K.t + K.h;
    S.hmin_cur = hmin_of(K.t);
    S.hmin_new = hmin_of(S.t_new);
    S.rem_new = P.t_max - S.t_new;
    return S;
}

// O3.3: clamp the step, detect the last step; called at t0 and after every accepted step
// (hmin, rem = hmin_of(K.t), t_max - K.t).
__device__ __forceinline__ void prepare_step(const KParams& P, Core& K, double hmin, double rem)
{
    double h = dmin(P.hmax, dmax(hmin, K.h));
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
    const double D[3] = {T.X[0] - T.X[3], T.X[1] - T.X[4], T.X[2] - T.X[5]};
    const double Xi[3] = {T.X[0], T.X[1], T.X[2]};
    accel<TRAP>(P, cs, D, Xi, T.A1, r2);
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
    prepare_step(P, K, hmin_of(K.t), P.t_max - K.t);
}

// Accept / reject logic of one attempt (O3.5-O3.8) on the controller state: err = the scaled
// error estimate, ST = step_times() of this attempt, (r2, s) = |d|^2 and d.u at the attempted step
// end.  Sets `accepted`; returns the stop status (>= 0) when the trajectory has ended, -1
// otherwise.  The caller moves ynew into y when `accepted` (also when the trajectory ends on this
// step).  `live` = false leaves everything untouched and returns -1 (lanes of the split kernel
// that hold no trajectory).
// Written without branches: both outcomes are formed and selected, so that the whole attempt is
// one basic block and the scheduler can hoist what depends on (t, h) only; the step-size chain
// behind the error estimate is what bounds the latency of a step.
template <class Cold>
__device__ __forceinline__ int finish_core(const KParams& P, Core& K, Cold& C, double err, const StepTimes& ST,
                                           double r2, double s, bool live, bool& accepted, bool& first_turn)
{
    const double q = err * P.inv_rtol;
    const double z = inv_fifth_root(q);  // (err/rtol)^(-1/5), for the reject path
    const bool acc = (err <= P.rtol);    // NaN rejects
    const unsigned fl = K.flags;
    const bool nofailed = (fl & kNoFailed) != 0u;
    const double h = K.h;
    // ---- accepted: observables, stop tests, next step size (O3.6-O3.8, O3.3).  What does not
    //      depend on z is formed first; behind z there is one product, one select, two clamps and
    //      the last-step test.
    const bool radial_min = (K.sprev < 0.0) & (s >= 0.0);
    const unsigned anymin = (fl & kAnyMin) | (radial_min ? kAnyMin : 0u);
    const bool counted = radial_min & (r2 < P.r_turn2);
    const int n_acc1 = K.n_acc + 1;
    const bool stop_exit = (anymin != 0u) & (r2 > P.r_exit2);
    const bool stop_last = (fl & kLast) != 0u;
    const bool stop_max = (long long)n_acc1 >= P.max_steps;
    const int st_acc = stop_exit ? 0 : (stop_last ? 1 : (stop_max ? 2 : -1));
    // h_cl = min(hmax, max(hmin_new, h_grow)) and last_new = (1.1 h_cl >= rem_new), with the three
    // comparisons of h_grow side by side instead of one behind the other (exact selects, same values)
    const double h_grown = grow_step(h, dmin(dmax(q, 1e-30), 1e30), fminf(fmaxf((float)q, 1e-30f), 1e30f));
    const double h_grow = nofailed ? h_grown : h;  // h is kept after a step with a failed attempt
    const bool over = (h_grow > P.hmax) | (ST.hmin_new > P.hmax);
    const bool under = (h_grow < ST.hmin_new);
    const bool last_grow = (1.1 * h_grow >= ST.rem_new);
    const bool last_max = (1.1 * P.hmax >= ST.rem_new), last_min = (1.1 * ST.hmin_new >= ST.rem_new);
    const double h_cl = over ? P.hmax : (under ? ST.hmin_new : h_grow);
    const bool last_new = over ? last_max : (under ? last_min : last_grow);
    const double h_acc = last_new ? ST.rem_new : h_cl;
    const unsigned fl_acc = anymin | kNoFailed | (last_new ? kLast : 0u);
    // ---- rejected: shrink (O3.5)
    const bool underflow = (h <= ST.hmin_cur);
    const double fac_z = (err == err) ? dmax(0.8 * z, 0.1) : 0.1;
    const double h_rej = dmax(h * (nofailed ? fac_z : 0.5), ST.hmin_cur);
    const int st_rej = underflow ? 3 : -1;
    // ---- commit
    const bool a = live & acc, r = live & !acc;
    accepted = a;
    if (Cold::kInRegisters) {
        C.rmin2() = (a & (r2 < C.rmin2())) ? r2 : C.rmin2();
        const bool c = a & counted;
        first_turn = c & (C.n_turn() == 0);
        C.t_first() = first_turn ? ST.t_new : C.t_first();
        C.t_last() = c ? ST.t_new : C.t_last();
        C.n_turn() += c ? 1 : 0;
        C.n_rej() += r ? 1 : 0;
    } else {
        first_turn = false;
        if (a) {
            if (r2 < C.rmin2()) C.rmin2() = r2;
            if (counted) {
                const int nt = ++C.n_turn();
                if (nt == 1) {
                    C.t_first() = ST.t_new;
                    first_turn = true;
                }
                C.t_last() = ST.t_new;
            }
        }
        if (r) C.n_rej()++;
    }
    K.n_acc = a ? n_acc1 : K.n_acc;
    K.t = a ? ST.t_new : K.t;
    K.sprev = a ? s : K.sprev;
    const bool keep = !live | (r & underflow) | (a & (st_acc >= 0));  // ended or idle: h, flags as they are
    K.h = keep ? h : (a ? h_acc : h_rej);
    K.flags = keep ? (a ? anymin | (fl & ~kAnyMin) : fl) : (a ? fl_acc : (fl & kAnyMin));
    return live ? (acc ? st_acc : st_rej) : -1;
}

// The common case of finish_core, for the six-lane integrator (whose step is bound by the instructions it
// issues): an accepted step with no failed attempt before it, no turning point, no stop, and a step size
// far above hmin.  fast_step_ok decides it from quantities that are known BEFORE the controller's fifth
// root (the warp votes on it while the root is being taken); fast_step_commit is then finish_core
// restricted to that case -- the same operations on the same operands, so the same bits:
//   * hmin = 16 ulp(t) <= 2^-48 |t|, and after an accepted step h_grow >= 0.79 h: with
//     h / 2 > 2^-48 |t_new| the clamps to hmin_new are no-ops (`under` false);
//   * h_grow <= 5 h (1 + 1e-6): with 5.5 h <= hmax and 1.1 x 5.5 h < t_max - t_new, `over` and `last_new`
//     are false: the next step size is h_grow itself and the flags do not change;
//   * no radial minimum this step: anymin = the flag as it is.
__device__ __forceinline__ bool fast_step_ok(const KParams& P, const Core& K, double q_own, double t_new, double r2,
                                             double s)
{
    // err = h max_k q_k <= rtol  <=>  h q_k <= rtol for every axis k (rounding is monotone): each lane tests
    // its own axis, the warp's vote combines them -- before the quotients have been gathered.  NaN fails.
    const bool acc_own = (K.h * q_own <= P.rtol);
    const bool finite_ok = (r2 > 0.0) & (r2 < 1.0e300) & (fabs(s) < 1.0e300);
    const unsigned fl = K.flags;
    const bool flags_ok = (fl & (kLast | kNoFailed)) == kNoFailed;
    const bool radial_min = (K.sprev < 0.0) & (s >= 0.0);
    const bool stop_exit = ((fl & kAnyMin) != 0u) & (r2 > P.r_exit2);
    const bool stop_max = (long long)(K.n_acc + 1) >= P.max_steps;
    // the next step size is at most 5 h (1 + 1e-6): with 5.5 h <= hmax and 1.1 x 5.5 h < t_max - t_new it is
    // neither clamped to hmax nor the last one; with h/2 > 2^-48 |t_new| >= hmin it is not clamped to hmin
    const double g = 5.5 * K.h;
    const bool h_ok = (g <= P.hmax) & (1.1 * g < P.t_max - t_new) & (K.h * 140737488355328.0 > fabs(t_new)) & (K.h > 1.0e-290);  // 2^47
    return acc_own & finite_ok & flags_ok & !radial_min & !stop_exit & !stop_max & h_ok;
}
template <class Cold>
__device__ __forceinline__ void fast_step_commit(const KParams& P, Core& K, Cold& C, double err, double t_new, double r2,
                                                 double s)
{
    const double q = err * P.inv_rtol;  // <= 1 here
    K.h = grow_step(K.h, q, (float)q);  // flags stay as they are: kNoFailed set, kLast not
    K.n_acc += 1;
    K.t = t_new;
    K.sprev = s;
    C.rmin2() = (r2 < C.rmin2()) ? r2 : C.rmin2();
}

// finish_core for the per-thread integrator: on return T holds the state to continue from (or
// the final state).  first_turn: this step counted the trajectory's first turning point (the
// "position" observable of PAPER.md:495 is the ion position T.X[0..2] at this moment).
template <class Cold>
__device__ __forceinline__ int finish_attempt(const KParams& P, Traj& T, Cold& C, const Attempt& R, bool& first_turn)
{
    bool accepted;
    const StepTimes ST = step_times(P, T.c);
    const int st = finish_core(P, T.c, C, R.err, ST, R.r2, R.s, true, accepted, first_turn);
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
