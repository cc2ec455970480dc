// aig_split.cuh -- one Dormand-Prince 5(4) step of ONE trajectory spread over SIX lanes of a warp.
//
// Why: a trajectory that forms a long-lived complex takes 10^2..10^3 times the mean number of steps
// (BASELINE.json north_star), and steps are sequential, so the run time of an
// ensemble is bounded below by (steps of the longest trajectory) x (latency of one step).  In the
// per-thread integrator a step is ~1200 warp instructions, 680 of them on the FP64 pipe (two cycles
// each): a warp cannot finish one in less than ~0.7 us however few of its lanes are alive, and takes
// ~3 us beside the eleven other warps of its SM (measured, profiles/r03_integrate_full.md).  Here the six
// lanes (k, e), k = x|y|z, e = 0|1 of a group hold component k of both particles and evaluate, at
// each of the three dependent levels of the Nystrom form, stage 2 lev + 2 + e; the per-lane
// instruction stream is ~3x shorter (422 instructions on the fast path) and a step costs about its
// dependent-chain latency: 0.64 us = 1,260 cycles measured (profiles/r02_integrate_full.md).
// Five groups share a warp (lanes 30, 31 idle).  The FP64 cost per trajectory step is ~2x that of
// the per-thread integrator (the scalar force factors, the controller and the step end are
// replicated), so only the few trajectories that outlive the step budget of the per-thread
// integrator are continued here.
//
// Arithmetic: identical to aig_device.cuh operation by operation (same scalar functions, same
// operand order in every cross-lane sum), so a trajectory's result does not depend on where it
// was continued.  The only formal difference: stage sums are padded to a common length with
// coefficient 0.0 (fma(0, A, acc) = acc exactly for finite A).
#pragma once
#include "aig_device.cuh"

#ifndef AIG_SPLIT_EARLY_RCP
#define AIG_SPLIT_EARLY_RCP 1
#endif

namespace aig {

constexpr int kGroupLanes = 6;                     // lanes per trajectory
constexpr int kGroupsPerWarp = 32 / kGroupLanes;   // 5

// What one lane holds of its trajectory: component k of both particles.
struct SplitState {
    double xi, vi, a1i;  // ion: position, velocity, acceleration at (t, y) (FSAL)
    double xa, va, a1a;  // atom
};

// Per-lane constants (registers): role in the group and the tableau entries of "my" stages.
struct SplitRole {
    int k, e, base;      // component, stage parity, first lane of my group
    bool ghost;          // lanes 30, 31: no trajectory, they only keep the shuffles convergent
    double cA0;          // level 0 (stage 2 | 3): coefficient of A_1
    double cA1[3];       // level 1 (stage 4 | 5): coefficients of A_1..A_3
    double cA2[5];       // level 2 (stage 6 | 7): coefficients of A_1..A_5
    double cC[3];        // c of my stage at each level
    double cCos;         // the cos this lane evaluates: at t + cCos h ...
    bool cos_end;        // ... or at t_new (stages 6, 7)
    double wa, wb;       // trap stiffness coefficients of axis k
};

__device__ __forceinline__ SplitRole make_role(const KParams& P)
{
    SplitRole R;
    const int lane = threadIdx.x & 31;
    const int g = lane / kGroupLanes, j = lane - g * kGroupLanes;
    R.ghost = (g >= kGroupsPerWarp);
    R.base = R.ghost ? (kGroupsPerWarp - 1) * kGroupLanes : g * kGroupLanes;  // ghosts mirror group 4's sources
    R.k = R.ghost ? 0 : (j >> 1);
    R.e = j & 1;
    const int e = R.e;
    R.cA0 = e ? kAbar[2][0] : 0.0;
#pragma unroll
    for (int l = 0; l < 3; ++l) R.cA1[l] = (l <= 1 + e) ? kAbar[3 + e][l] : 0.0;
#pragma unroll
    for (int l = 0; l < 5; ++l) R.cA2[l] = (l <= 3 + e) ? kAbar[5 + e][l] : 0.0;
#pragma unroll
    for (int lev = 0; lev < 3; ++lev) R.cC[lev] = kC[2 * lev + 1 + e];
    const int jj = R.ghost ? 0 : j;
    R.cCos = kC[jj + 1];
    R.cos_end = (jj >= 4);
    R.wa = P.wa[R.k];
    R.wb = P.wb[R.k];
    return R;
}

// Result of one attempted step as seen by one lane.
struct SplitAttempt {
    SplitState Y;              // ynew (component k) and f(t_new, ynew)
    double t_new, err, r2, s;  // as in Attempt, except: err = the raw estimate, to be replaced by NaN when !finite
    double q_own;              // this lane's axis quotient (err = h max over the three axes)
    bool finite;
};

__device__ __forceinline__ double shfl_d(double v, int src) { return __shfl_sync(0xffffffffu, v, src); }
__device__ __forceinline__ double shfl_xor_d(double v, int m) { return __shfl_xor_sync(0xffffffffu, v, m); }

// One level in two halves, in the order the dependent chain runs:
//   level_open : position of my stage from the accelerations known so far, d_k^2, and the three
//                shuffles that gather |d|^2 over k are issued;
//   level_close: 1/r^2 -> force factors -> accelerations -> exchange with the partner lane (k, 1 - e).
// Whatever the caller puts between the two (the cos of this step, the partial step-end sums)
// runs inside the shuffle latency.
struct LevelOpen {
    double xsi, xsa, d;  // ion stage position, atom stage position (level 2 only: the new state), relative position
    double s0, s1, s2;
};
template <int LEV>
__device__ __forceinline__ void level_open(const SplitRole& R, const SplitState& Y, double d0, double u0, double h,
                                           double h2, const double (&Ai)[7], const double (&Aa)[7], LevelOpen& L)
{
    const double hc = h * R.cC[LEV];
    double acci, acca;
    if (LEV == 0) {
        acci = R.cA0 * Ai[0];
        acca = R.cA0 * Aa[0];
    } else if (LEV == 1) {
        acci = R.cA1[0] * Ai[0];
        acca = R.cA1[0] * Aa[0];
#pragma unroll
        for (int l = 1; l < 3; ++l) {
            acci = fma(R.cA1[l], Ai[l], acci);
            acca = fma(R.cA1[l], Aa[l], acca);
        }
    } else {
        acci = R.cA2[0] * Ai[0];
        acca = R.cA2[0] * Aa[0];
#pragma unroll
        for (int l = 1; l < 5; ++l) {
            acci = fma(R.cA2[l], Ai[l], acci);
            acca = fma(R.cA2[l], Aa[l], acca);
        }
    }
    // the same three chains as dp45_attempt (aig_device.cuh "Stage positions"); stage 2 (level 0, e = 0) has
    // coefficient 0: acc = +-0 and fma(h2, +-0, base) = base exactly
    L.xsi = stage_pos(Y.xi, Y.vi, hc, h2, acci);
    L.d = stage_pos(d0, u0, hc, h2, acci - acca);
    L.xsa = (LEV == 2) ? stage_pos(Y.xa, Y.va, hc, h2, acca) : 0.0;
    const double sq = L.d * L.d;
    const int src = R.base + R.e;
    L.s0 = shfl_d(sq, src);
    L.s1 = shfl_d(sq, src + 2);
    L.s2 = shfl_d(sq, src + 4);
}
template <int TRAP, int LEV>
__device__ __forceinline__ double level_close(const KParams& P, const SplitRole& R, const LevelOpen& L,
                                              double mycos, double (&Ai)[7], double (&Aa)[7])
{
    double trap = 0.0;
    if (trap_of(TRAP) != TRAP_NONE) {
        const double cs = (trap_of(TRAP) == TRAP_STATIC) ? 1.0 : shfl_d(mycos, R.base + 2 * LEV + R.e);
        trap = -(trap_w<TRAP>(R.wa, R.wb, cs) * L.xsi);
    }
    const double r2 = sum3(L.s0, L.s1, L.s2);
    double gi, ga;
    force_factors<TRAP>(P, r2, gi, ga);
    const double myAa = ga * L.d;
    const double myAi = (trap_of(TRAP) == TRAP_NONE) ? gi * L.d : fma(gi, L.d, trap);
    const double pAi = shfl_xor_d(myAi, 1);
    const double pAa = shfl_xor_d(myAa, 1);
    Ai[2 * LEV + 1] = R.e ? pAi : myAi;
    Ai[2 * LEV + 2] = R.e ? myAi : pAi;
    Aa[2 * LEV + 1] = R.e ? pAa : myAa;
    Aa[2 * LEV + 2] = R.e ? myAa : pAa;
    return r2;
}

// One attempted step of size K.h from (K.t, y) for every group of the warp.  All 32 lanes call it
// together (full-mask shuffles); lanes without a trajectory run it on benign dummy state.
template <int TRAP>
__device__ __forceinline__ void split_attempt(const KParams& P, const SplitRole& R, const Core& K,
                                              const SplitState& Y, SplitAttempt& out)
{
    const double h = K.h;
    const double h2 = h * h;
    const double t_new = (K.flags & kLast) ? P.t_max : K.t + h;
    double Ai[7], Aa[7];
    Ai[0] = Y.a1i;
    Aa[0] = Y.a1a;
    const double d0 = Y.xi - Y.xa, u0 = Y.vi - Y.va;  // relative position and velocity at the beginning of the step
    LevelOpen L;
    level_open<0>(R, Y, d0, u0, h, h2, Ai, Aa, L);
    // the cos of my stage time, inside the first level's shuffle and reciprocal latency
    double mycos = 1.0;
    if (trap_of(TRAP) == TRAP_RF || trap_of(TRAP) == TRAP_RF_BIG) mycos = trap_cos<TRAP>(P, R.cos_end ? t_new : fma(R.cCos, h, K.t));
    level_close<TRAP, 0>(P, R, L, mycos, Ai, Aa);
    level_open<1>(R, Y, d0, u0, h, h2, Ai, Aa, L);
    level_close<TRAP, 1>(P, R, L, mycos, Ai, Aa);
    level_open<2>(R, Y, d0, u0, h, h2, Ai, Aa, L);
    // everything of the step end that does not need stages 6 and 7 goes inside the last level
    StepEndPart Si, Sa;
    step_end_begin(P, Y.xi, Y.vi, Ai, Si);
    step_end_begin(P, Y.xa, Y.va, Aa, Sa);
    const double r2 = level_close<TRAP, 2>(P, R, L, mycos, Ai, Aa);
    const double xsi = L.xsi, xsa = L.xsa;
    // stage 7 (lanes e = 1) is the 5th-order solution: hand x_new and |d|^2 there to the partner
    const double pxi = shfl_xor_d(xsi, 1), pxa = shfl_xor_d(xsa, 1), pr2 = shfl_xor_d(r2, 1);
    const double xni = R.e ? xsi : pxi, xna = R.e ? xsa : pxa;
    out.r2 = R.e ? r2 : pr2;
    // step end of component k of both particles (replicated on both lanes of the pair)
    Ratio cvi, cxi, cva, cxa;
    const double vni = step_end_finish(Si, h, xni, Y.vi, Ai[5], Ai[6], cvi, cxi);
    const double vna = step_end_finish(Sa, h, xna, Y.va, Aa[5], Aa[6], cva, cxa);
    const double q = AIG_SPLIT_EARLY_RCP ? axis_quotient_early_rcp(cvi, cxi, cva, cxa) : axis_quotient(cvi, cxi, cva, cxa);
    const double p = (xna - xni) * (vna - vni);
    const int src = R.base + R.e;
    const double q0 = shfl_d(q, src), q1 = shfl_d(q, src + 2), q2 = shfl_d(q, src + 4);
    const double p0 = shfl_d(p, src), p1 = shfl_d(p, src + 2), p2 = shfl_d(p, src + 4);
    out.s = sum3(p0, p1, p2);
    out.t_new = t_new;
    out.q_own = q;
    out.err = error_raw(h, q0, q1, q2);
    out.finite = attempt_finite(q0, q1, q2, out.r2, out.s);
    out.Y.xi = xni;
    out.Y.vi = vni;
    out.Y.a1i = Ai[6];
    out.Y.xa = xna;
    out.Y.va = vna;
    out.Y.a1a = Aa[6];
}

}  // namespace aig
