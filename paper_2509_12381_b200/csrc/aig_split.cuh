// aig_split.cuh -- one Dormand-Prince 5(4) step of ONE trajectory spread over SIX lanes of a warp.
//
// Why: a trajectory that forms a long-lived complex takes 10^2..10^3 times the mean number of steps
// (BASELINE.json north_star), and steps are sequential, so the run time of an
// ensemble is bounded below by (steps of the longest trajectory) x (latency of one step).  In the
// per-thread integrator a step is ~1100 warp instructions, ~600 of them on the half-rate FP64 pipe:
// a warp cannot finish one in less than ~1.2 us however few of its lanes are alive.  Here the six
// lanes (k, e), k = x|y|z, e = 0|1 of a group hold component k of both particles and evaluate, at
// each of the three dependent levels of the Nystrom form, stage 2 lev + 2 + e; the per-lane
// instruction stream is ~4x shorter and a step costs about its dependent-chain latency (~0.5 us).
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
    double t_new, err, r2, s;  // as in Attempt
};

__device__ __forceinline__ double shfl_d(double v, int src) { return __shfl_sync(0xffffffffu, v, src); }
__device__ __forceinline__ double shfl_xor_d(double v, int m) { return __shfl_xor_sync(0xffffffffu, v, m); }

// One level: position of my stage from the accelerations known so far, the force there, and the
// exchange with the partner lane (k, 1 - e).  NT = number of stage accelerations in the sum.
template <int TRAP, int LEV>
__device__ __forceinline__ void split_level(const KParams& P, const SplitRole& R, const SplitState& Y, double h,
                                            double h2, double mycos, double (&Ai)[7], double (&Aa)[7],
                                            double& xsi, double& xsa, double& r2)
{
    const double cs = (TRAP == TRAP_RF || TRAP == TRAP_RF_BIG) ? shfl_d(mycos, R.base + 2 * LEV + R.e) : 1.0;
    const double hc = h * R.cC[LEV];
    const double bi = fma(hc, Y.vi, Y.xi);
    const double ba = fma(hc, Y.va, Y.xa);
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
    xsi = fma(h2, acci, bi);
    xsa = fma(h2, acca, ba);
    const double d = xsi - xsa;
    const double sq = d * d;
    const int src = R.base + R.e;
    r2 = sum3(shfl_d(sq, src), shfl_d(sq, src + 2), shfl_d(sq, src + 4));
    double gi, ga;
    force_factors(P, r2, gi, ga);
    const double myAa = ga * d;
    const double myAi = (TRAP == TRAP_NONE) ? gi * d : fma(-trap_w<TRAP>(R.wa, R.wb, cs), xsi, gi * d);
    const double pAi = shfl_xor_d(myAi, 1);
    const double pAa = shfl_xor_d(myAa, 1);
    Ai[2 * LEV + 1] = R.e ? pAi : myAi;
    Ai[2 * LEV + 2] = R.e ? myAi : pAi;
    Aa[2 * LEV + 1] = R.e ? pAa : myAa;
    Aa[2 * LEV + 2] = R.e ? myAa : pAa;
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
    double mycos = 1.0;
    if (TRAP == TRAP_RF || TRAP == TRAP_RF_BIG) mycos = trap_cos<TRAP>(P, R.cos_end ? t_new : fma(R.cCos, h, K.t));
    double Ai[7], Aa[7];
    Ai[0] = Y.a1i;
    Aa[0] = Y.a1a;
    double xsi, xsa, r2;
    split_level<TRAP, 0>(P, R, Y, h, h2, mycos, Ai, Aa, xsi, xsa, r2);
    split_level<TRAP, 1>(P, R, Y, h, h2, mycos, Ai, Aa, xsi, xsa, r2);
    split_level<TRAP, 2>(P, R, Y, h, h2, mycos, Ai, Aa, xsi, xsa, r2);
    // stage 7 (lanes e = 1) is the 5th-order solution: hand x_new and |d|^2 there to the partner
    const double pxi = shfl_xor_d(xsi, 1), pxa = shfl_xor_d(xsa, 1), pr2 = shfl_xor_d(r2, 1);
    const double xni = R.e ? xsi : pxi, xna = R.e ? xsa : pxa;
    out.r2 = R.e ? r2 : pr2;
    // step end of component k of both particles (replicated on both lanes of the pair)
    Ratio cvi, cxi, cva, cxa;
    const double vni = step_end_component(P, h, Y.xi, xni, Y.vi, Ai, cvi, cxi);
    const double vna = step_end_component(P, h, Y.xa, xna, Y.va, Aa, cva, cxa);
    const Ratio ai = ratio_max(cvi, cxi), aa = ratio_max(cva, cxa);
    const int src = R.base + R.e;
    Ratio gi3[3], ga3[3];
#pragma unroll
    for (int m = 0; m < 3; ++m) {
        gi3[m].n = shfl_d(ai.n, src + 2 * m);
        gi3[m].d = shfl_d(ai.d, src + 2 * m);
        ga3[m].n = shfl_d(aa.n, src + 2 * m);
        ga3[m].d = shfl_d(aa.d, src + 2 * m);
    }
    const Ratio ion = ratio_max(ratio_max(gi3[0], gi3[1]), gi3[2]);
    const Ratio atom = ratio_max(ratio_max(ga3[0], ga3[1]), ga3[2]);
    const double p = (xna - xni) * (vna - vni);
    out.s = sum3(shfl_d(p, src), shfl_d(p, src + 2), shfl_d(p, src + 4));
    out.t_new = t_new;
    out.err = error_estimate(h, ion, atom, out.r2, out.s);
    out.Y.xi = xni;
    out.Y.vi = vni;
    out.Y.a1i = Ai[6];
    out.Y.xa = xna;
    out.Y.va = vna;
    out.Y.a1a = Aa[6];
}

}  // namespace aig
