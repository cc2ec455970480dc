// aig_kernels.cu -- kernels and C ABI of libaig (include/aig.h).  sm_100a only.
//
// Kernels
//   plan_*_kernel            : order the work queue in three classes: slow capture candidates (impact
//                              parameter inside 1.5 Langevin radii: the only ones that can form a
//                              long-lived complex; the slow ones last longest), the other candidates,
//                              the rest.  Scheduling only.
//   integrate_kernel<TRAP>   : persistent threads, one trajectory per lane, registers only;
//                              finished lanes refill from a global atomic work queue
//                              (warp-aggregated: one atomicAdd per warp per refill event); a
//                              trajectory that outlives the step budget is suspended into a
//                              checkpoint slot.
//   integrate_split_kernel<TRAP> : continues suspended trajectories, six lanes per trajectory
//                              (aig_split.cuh): half the step latency, for the long-lived tail.
//   step_once_kernel<TRAP>   : test hook, one attempted step per thread.
//   histogram_kernel         : shared-memory privatised bins, warp-aggregated increments.
//   dfma_probe_kernel        : FP64 FMA chains, measures the non-tensor FP64 roofline.
//
// Nothing here is a dense contraction: no tensor cores, no TMA.  The bound is the FP64 pipe;
// global memory sees 96 B in and ~150 B out per trajectory against ~1e5 flops.
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <algorithm>
#include <atomic>
#include <cstdlib>
#include <mutex>
#include <cuda_runtime.h>

#include "../../include/aig.h"
#include "aig_device.cuh"
#include "aig_split.cuh"

namespace aig {

#ifndef AIG_BLOCK
#define AIG_BLOCK 128
#endif
#ifndef AIG_MIN_BLOCKS
#define AIG_MIN_BLOCKS 2
#endif
#ifndef AIG_SPLIT_UNROLL
#define AIG_SPLIT_UNROLL 2
#endif
constexpr int kSplitUnroll = AIG_SPLIT_UNROLL;  // steps per basic block of the six-lane integrator
constexpr int kBlock = AIG_BLOCK;             // threads per block of the integrator
constexpr int kBlocksPerSM = AIG_MIN_BLOCKS;  // resident blocks per SM the register budget is sized for

// Stage timeline (diagnostics): counters[kCntTime + 2 s] = %globaltimer when block 0 of stage s started,
// counters[kCntTime + 2 s + 1] = latest %globaltimer at which one of its blocks ended (ns).
constexpr int kCntTime = 32;
__device__ __forceinline__ unsigned long long global_ns()
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
    return t;
}
__device__ __forceinline__ void stage_begin(unsigned long long* tl)
{
    if (tl && blockIdx.x == 0 && threadIdx.x == 0) tl[0] = global_ns();
}
__device__ __forceinline__ void stage_end(unsigned long long* tl)
{
    if (tl && (threadIdx.x & 31) == 0) atomicMax(tl + 1, global_ns());
}

struct OutPtrs {
    double *y_final, *t_final, *lifetime, *angle, *r_min;
    int *n_acc, *n_rej, *n_turn, *status;
    unsigned char* complex_flag;
    double* x_turn1;  // [3][N] ion position at the first counted turning point, or nullptr (not recorded)
};

// ------------------------------------------------------------------------------------------
// integrator
// ------------------------------------------------------------------------------------------
// Cold state of the per-thread integrator: one shared-memory slot per thread, SoA (conflict-free).
struct ColdShared {
    static constexpr bool kInRegisters = false;
    __device__ __forceinline__ double& rmin2() { return s_rmin2[threadIdx.x]; }
    __device__ __forceinline__ double& t_first() { return s_tfirst[threadIdx.x]; }
    __device__ __forceinline__ double& t_last() { return s_tlast[threadIdx.x]; }
    __device__ __forceinline__ int& n_rej() { return s_nrej[threadIdx.x]; }
    __device__ __forceinline__ int& n_turn() { return s_nturn[threadIdx.x]; }
    double* s_rmin2;
    double* s_tfirst;
    double* s_tlast;
    int* s_nrej;
    int* s_nturn;
};

template <int TRAP, class Cold>
__device__ __forceinline__ void load_traj(const KParams& P, const double* __restrict__ y0,
                                          long long N, long long idx, Traj& T, Cold& C)
{
    // rows of y0: 0-2 ion position, 3-5 ion velocity, 6-8 atom position, 9-11 atom velocity
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        T.X[k] = __ldg(y0 + (0 + k) * N + idx);
        T.V[k] = __ldg(y0 + (3 + k) * N + idx);
        T.X[3 + k] = __ldg(y0 + (6 + k) * N + idx);
        T.V[3 + k] = __ldg(y0 + (9 + k) * N + idx);
    }
    init_traj<TRAP>(P, T, C);
}

// scalar observables of a finished trajectory (a8); v0 / v1 = initial / final atom velocity
template <class Cold>
__device__ __forceinline__ void store_scalars(long long idx, const Core& K, Cold& C, int status,
                                              const double (&v0)[3], const double (&v1)[3], const OutPtrs& O)
{
    O.t_final[idx] = K.t;
    O.angle[idx] = angle_between(v0, v1);
    O.r_min[idx] = sqrt(C.rmin2());
    const int n_turn = C.n_turn();
    const bool cplx = n_turn >= 2;
    O.lifetime[idx] = cplx ? C.t_last() - C.t_first() : 0.0;
    O.n_acc[idx] = K.n_acc;
    O.n_rej[idx] = C.n_rej();
    O.n_turn[idx] = n_turn;
    O.status[idx] = status;
    O.complex_flag[idx] = cplx ? 1 : 0;
}

template <class Cold>
__device__ __forceinline__ void store_traj(const double (&v0)[3], long long N, long long idx,
                                           const Traj& T, Cold& C, int status, const OutPtrs& O)
{
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        O.y_final[(0 + k) * N + idx] = T.X[k];
        O.y_final[(3 + k) * N + idx] = T.V[k];
        O.y_final[(6 + k) * N + idx] = T.X[3 + k];
        O.y_final[(9 + k) * N + idx] = T.V[3 + k];
    }
    const double v1[3] = {T.V[3], T.V[4], T.V[5]};
    store_scalars(idx, T.c, C, status, v0, v1, O);
}

// Checkpoint slots: the full state of a suspended trajectory, SoA over `cap` slots
// (d: 24 doubles per slot, i: 4 ints, idx: the trajectory's global index).
//   d rows: 0-2 x_ion, 3-5 x_atom, 6-8 v_ion, 9-11 v_atom, 12-14 a_ion, 15-17 a_atom (FSAL),
//           18 t, 19 h, 20 s(t), 21 r_min^2, 22 t_first, 23 t_last;  i rows: n_acc, flags, n_rej, n_turn
struct Ckpt {
    double* d;
    int* i;
    long long* idx;
    long long cap;
};
constexpr int kCkptDoubles = 24, kCkptInts = 4;
constexpr size_t kCkptBytesPerSlot = kCkptDoubles * 8 + kCkptInts * 4 + 8;

template <class Cold>
__device__ __forceinline__ void ckpt_store(const Ckpt& K, long long slot, long long idx, const Traj& T, Cold& C)
{
    double* d = K.d + slot;
    const size_t cap = (size_t)K.cap;
#pragma unroll
    for (int j = 0; j < 6; ++j) {
        d[(0 + j) * cap] = T.X[j];
        d[(6 + j) * cap] = T.V[j];
        d[(12 + j) * cap] = T.A1[j];
    }
    d[18 * cap] = T.c.t;
    d[19 * cap] = T.c.h;
    d[20 * cap] = T.c.sprev;
    d[21 * cap] = C.rmin2();
    d[22 * cap] = C.t_first();
    d[23 * cap] = C.t_last();
    int* q = K.i + slot;
    q[0 * cap] = T.c.n_acc;
    q[1 * cap] = (int)T.c.flags;
    q[2 * cap] = C.n_rej();
    q[3 * cap] = C.n_turn();
    K.idx[slot] = idx;
}

// Scheduling arguments of one launch of the per-thread integrator.  Work items are the entries
// [*begin, *end) of `order` (trajectory indices; order == nullptr: the indices themselves).  A lane
// whose trajectory has not ended is suspended (state written to slot atomicAdd(*n_out, 1) of
// `out`) when it has taken `budget` accepted steps -- as long as this stage has handed over fewer
// than `soft_cap` trajectories (the six-lane integrator has half the throughput per FP64
// operation: it is for the few, not for the many; a trajectory that is kept is asked again one
// budget later), and only once it is `mean_factor` times longer than the mean of the trajectories
// this launch has finished (a workload where every trajectory is long is the per-thread kernel's
// job: nothing is handed over before 32 have finished) -- or when, `tail_iters` iterations after its
// warp has seen the queue empty, the warp has `drain_lanes` or fewer trajectories left; when the
// slots are exhausted it simply keeps stepping.  Suspension never changes a trajectory's
// arithmetic, only where it continues.
struct Sched {
    unsigned long long* queue;
    const long long* order;
    const unsigned long long *begin, *end;
    unsigned long long* n_out;
    const unsigned long long* soft_base;  // slots handed out before this stage
    long long soft_cap;
    Ckpt out;
    int budget;
    int tail_iters;
    int refill_batch, refill_wait;
    int drain_lanes;            // after the queue ran dry a warp hands its trajectories over once it has this few left
    unsigned long long* stats;  // [0] accepted steps, [1] number of the trajectories this launch has finished
    int mean_factor;            // hand over only beyond mean_factor x their mean (0: the plain budget)
    unsigned long long* timeline;
};

template <int TRAP, int BLOCK, int MINB>
__global__ void __launch_bounds__(BLOCK, MINB)
integrate_kernel(const KParams P, const double* __restrict__ y0, const long long N, const OutPtrs O,
                 const Sched S)
{
    __shared__ double s_rmin2[BLOCK], s_tfirst[BLOCK], s_tlast[BLOCK];
    __shared__ double s_v0[3][BLOCK];  // initial atom velocity (for the scattering angle at the end)
    __shared__ int s_nrej[BLOCK], s_nturn[BLOCK];
    ColdShared C{s_rmin2, s_tfirst, s_tlast, s_nrej, s_nturn};
    const unsigned FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    const long long first = (long long)*S.begin;
    const long long total = (long long)*S.end - first;
    const long long soft_first = (long long)*S.soft_base;
    Traj T;
    long long idx = -1;
    int stop_at = 0;      // suspend when n_acc reaches this
    int since_dry = 0;    // warp-uniform: iterations since the queue was seen empty
    bool live = false;
    bool dry = false;     // warp-uniform: the queue has been seen empty
    bool may_suspend = true;
    int pending = -1;     // stop status of a finished trajectory whose results are not stored yet
    int waited = 0;       // warp-uniform: iterations since a lane of this warp went idle
    stage_begin(S.timeline);

    for (;;) {
        // ---- service: lanes without a trajectory store what they finished and take the next items
        //      of the queue.  The whole warp walks through this code (atan2 / sqrt of the end, global
        //      loads and the twelve divisions of the start) whenever one lane needs it, so idle lanes
        //      are served in batches: when refill_batch of them wait, or one has waited refill_wait
        //      iterations, or the queue is empty.
        const unsigned need = __ballot_sync(FULL, !live);
        if (need && (__popc(need) >= S.refill_batch || waited >= S.refill_wait || dry)) {
            waited = 0;
            {   // accepted steps and count of what this warp has finished since its last service
                const unsigned fm = __ballot_sync(FULL, pending >= 0);
                if (fm) {
                    const unsigned steps = __reduce_add_sync(FULL, pending >= 0 ? (unsigned)T.c.n_acc : 0u);
                    if (lane == 0) {
                        atomicAdd(S.stats + 0, (unsigned long long)steps);
                        atomicAdd(S.stats + 1, (unsigned long long)__popc(fm));
                    }
                }
            }
            if (pending >= 0) {
                const double v0[3] = {s_v0[0][threadIdx.x], s_v0[1][threadIdx.x], s_v0[2][threadIdx.x]};
                store_traj(v0, N, idx, T, C, pending, O);
                pending = -1;
            }
            if (!dry) {
                const int cnt = __popc(need);
                const int leader = __ffs(need) - 1;
                unsigned long long base = 0;
                if (lane == leader) base = atomicAdd(S.queue, (unsigned long long)cnt);
                base = __shfl_sync(FULL, base, leader);
                if (!live) {
                    const long long cand = (long long)base + __popc(need & ((1u << lane) - 1u));
                    if (cand < total) {
                        idx = S.order ? S.order[first + cand] : first + cand;
                        load_traj<TRAP>(P, y0, N, idx, T, C);
#pragma unroll
                        for (int k = 0; k < 3; ++k) s_v0[k][threadIdx.x] = T.V[3 + k];
                        stop_at = S.budget;
                        may_suspend = true;
                        live = true;
                    }
                }
                if ((long long)base + cnt >= total) dry = true;
            }
            if (!__any_sync(FULL, live)) break;
        } else if (need) {
            ++waited;
        }
        // warp-uniform: the queue is empty, the grace period is over and few lanes are still alive: at
        // fewer than ~11 lanes the six-lane kernel does more steps per SM and second than this one
        const bool drain = dry && since_dry > S.tail_iters && (32 - __popc(need)) <= S.drain_lanes;
        if (dry) ++since_dry;
        // ---- one attempted step for every live lane
        if (live) {
            Attempt R;
            dp45_attempt<TRAP>(P, T, R);
            bool first_turn;
            const int st = finish_attempt(P, T, C, R, first_turn);
            if (first_turn && O.x_turn1) {  // once per trajectory ("position")
#pragma unroll
                for (int k = 0; k < 3; ++k) O.x_turn1[k * N + idx] = T.X[k];
            }
            if (st >= 0) {
                pending = st;
                live = false;
            } else if (may_suspend && (T.c.n_acc >= stop_at || drain)) {
                bool room = true;
                if (!drain) {
                    // budget hand-over: only while the six-lane queue is short, and only for a trajectory
                    // that is long compared with what this launch has finished so far
                    const long long used = (long long)(*(volatile unsigned long long*)S.n_out) - soft_first;
                    room = used < S.soft_cap;
                    if (room && S.mean_factor > 0) {
                        const unsigned long long cnt = *(volatile unsigned long long*)(S.stats + 1);
                        const unsigned long long sum = *(volatile unsigned long long*)(S.stats + 0);
                        room = (cnt >= 32ULL) && ((unsigned long long)T.c.n_acc * cnt >= (unsigned long long)S.mean_factor * sum);
                    }
                    if (!room) stop_at += S.budget;
                }
                if (room) {
                    const long long slot = (long long)atomicAdd(S.n_out, 1ULL);
                    if (slot < S.out.cap) {
                        ckpt_store(S.out, slot, idx, T, C);
                        live = false;
                    } else {
                        may_suspend = false;  // no slot left: finish it here
                    }
                }
            }
        }
    }
    stage_end(S.timeline);
}

// ---- six lanes per trajectory: continues the slots [*begin, min(*end, cap)) of `in` to their end
// nq queues, served in this order: the pass's own slot range first, then the ranges of the stages
// before it (their bulk passes are complete, so their slots are too): a pass that runs out of work
// helps drain what an earlier, smaller pass is still working through.
struct SplitSched {
    unsigned long long* timeline;
    unsigned long long* loaded;  // diagnostics: trajectories this pass has taken
    int nq;
    unsigned long long* queue[4];
    const unsigned long long *begin[4], *end[4];
    Ckpt in;
};

template <int TRAP, int WARPS, int MINB>
__global__ void __launch_bounds__(32 * WARPS, MINB)
integrate_split_kernel(const KParams P, const double* __restrict__ y0, const long long N, const OutPtrs O,
                       const SplitSched S)
{
    const unsigned FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    const SplitRole R = make_role(P);
    const bool leader = !R.ghost && (lane == R.base);
    int qi = 0;  // warp-uniform: the queue being served
    long long first = 0, total = 0;
    auto open_queue = [&]() {
        const unsigned long long e = *S.end[qi];
        first = (long long)*S.begin[qi];
        total = (long long)(e < (unsigned long long)S.in.cap ? e : (unsigned long long)S.in.cap) - first;
    };
    open_queue();
    // benign state for lanes without a trajectory (they take part in every shuffle)
    SplitState Y;
    Y.xi = 1.0 + R.k;
    Y.xa = 101.0 + 2.0 * R.k;
    Y.vi = Y.va = Y.a1i = Y.a1a = 0.0;
    Core K;
    K.t = P.t0;
    K.h = 1.0;
    K.sprev = 0.0;
    K.n_acc = 0;
    K.flags = 0u;
    ColdRegs C;
    C.rmin2_ = C.t_first_ = C.t_last_ = 0.0;
    C.n_rej_ = C.n_turn_ = 0;
    long long idx = -1;
    bool live = false;
    bool dry = false;  // warp-uniform: every queue has been seen empty

    // refill: every idle group takes the next slot of the queue (one atomicAdd per warp)
    auto refill_once = [&]() -> bool {   // returns true when another round may place more groups
        const unsigned need = __ballot_sync(FULL, leader && !live);
        if (need == 0u || dry) return false;
        while (total <= 0) {  // skip empty ranges
            if (++qi >= S.nq) {
                dry = true;
                return false;
            }
            open_queue();
        }
        const int cnt = __popc(need);
        unsigned long long base = 0;
        if (lane == 0) base = atomicAdd(S.queue[qi], (unsigned long long)cnt);
        base = __shfl_sync(FULL, base, 0);
        if (lane == 0) {
            const long long got = total - (long long)base;
            if (got > 0) atomicAdd(S.loaded, (unsigned long long)(got < cnt ? got : cnt));
        }
        if (!R.ghost && ((need >> R.base) & 1u)) {
            const long long cand = (long long)base + __popc(need & ((1u << R.base) - 1u));
            if (cand < total) {
                const long long slot = first + cand;
                const size_t cap = (size_t)S.in.cap;
                const double* d = S.in.d + slot;
                Y.xi = d[(0 + R.k) * cap];
                Y.xa = d[(3 + R.k) * cap];
                Y.vi = d[(6 + R.k) * cap];
                Y.va = d[(9 + R.k) * cap];
                Y.a1i = d[(12 + R.k) * cap];
                Y.a1a = d[(15 + R.k) * cap];
                K.t = d[18 * cap];
                K.h = d[19 * cap];
                K.sprev = d[20 * cap];
                C.rmin2_ = d[21 * cap];
                C.t_first_ = d[22 * cap];
                C.t_last_ = d[23 * cap];
                const int* q = S.in.i + slot;
                K.n_acc = q[0 * cap];
                K.flags = (unsigned)q[1 * cap];
                C.n_rej_ = q[2 * cap];
                C.n_turn_ = q[3 * cap];
                idx = S.in.idx[slot];
                live = true;
            }
        }
        if ((long long)base + cnt >= total) {  // this range is exhausted: go on with the next one
            if (++qi >= S.nq) {
                dry = true;
                return false;
            }
            open_queue();
            return true;
        }
        return false;
    };
    auto refill = [&]() {
        while (refill_once()) {
        }
    };

    stage_begin(S.timeline);
    refill();
    if (!__any_sync(FULL, live)) {
        stage_end(S.timeline);
        return;
    }
    for (;;) {
        // ---- kSplitUnroll attempted steps for every group (all lanes together: full-mask shuffles
        //      inside), straight-line code up to the vote below.  Several steps per basic block
        //      because the step-size chain of one step continues into the next: the instruction
        //      scheduler then sees it as the long path and orders a step's bookkeeping (state
        //      selects, observables, stop tests) behind it instead of in front of it.  A group whose
        //      trajectory ends inside the block idles for the rest of it (st keeps the status).
        int st = -1;
#pragma unroll
        for (int u = 0; u < kSplitUnroll; ++u) {
            SplitAttempt A;
            StepTimes ST;
            split_attempt<TRAP>(P, R, K, Y, A, ST);
            bool accepted, first_turn;
            const int s1 = finish_core(P, K, C, A.err, ST, A.r2, A.s, live & (st < 0), accepted, first_turn);
            // once per trajectory ("position"): lane (k, 0) holds component k of the ion
            if (first_turn && R.e == 0 && O.x_turn1) O.x_turn1[R.k * N + idx] = A.Y.xi;
            Y.xi = accepted ? A.Y.xi : Y.xi;
            Y.vi = accepted ? A.Y.vi : Y.vi;
            Y.a1i = accepted ? A.Y.a1i : Y.a1i;
            Y.xa = accepted ? A.Y.xa : Y.xa;
            Y.va = accepted ? A.Y.va : Y.va;
            Y.a1a = accepted ? A.Y.a1a : Y.a1a;
            st = (st < 0) ? s1 : st;
        }
        const unsigned fin = __ballot_sync(FULL, st >= 0);
        if (fin == 0u) continue;
        // ---- a8 (rare): lanes e = 0 store component k of the final state, the group's first lane
        //      the scalars; then the group takes the next slot
        if (st >= 0) {
            const double v1[3] = {__shfl_sync(fin, Y.va, R.base), __shfl_sync(fin, Y.va, R.base + 2),
                                  __shfl_sync(fin, Y.va, R.base + 4)};
            if (R.e == 0) {
                O.y_final[(0 + R.k) * N + idx] = Y.xi;
                O.y_final[(3 + R.k) * N + idx] = Y.vi;
                O.y_final[(6 + R.k) * N + idx] = Y.xa;
                O.y_final[(9 + R.k) * N + idx] = Y.va;
            }
            if (leader) {
                const double v0[3] = {__ldg(y0 + 9 * N + idx), __ldg(y0 + 10 * N + idx), __ldg(y0 + 11 * N + idx)};
                store_scalars(idx, K, C, st, v0, v1, O);
            }
            live = false;
            // benign state again: the idle group keeps stepping (untouched by finish_core) until it is refilled
            Y.xi = 1.0 + R.k;
            Y.xa = 101.0 + 2.0 * R.k;
            Y.vi = Y.va = Y.a1i = Y.a1a = 0.0;
            K.t = P.t0;
            K.h = 1.0;
            K.flags = 0u;
        }
        refill();
        if (!__any_sync(FULL, live)) break;
    }
    stage_end(S.timeline);
}

// ---- work-queue order: the trajectories that can become long first ------------------------------
// (1) A trajectory can only form a complex (orders of magnitude more steps) if it gets over the
//     centrifugal barrier of the -C4/r^4 tail, i.e. if its impact parameter b is below the
//     Langevin radius b_c = (4 C4/E)^(1/4), E = mu u^2/2 (relative motion at t0): "candidates" are
//     those with b < kappa b_c (kappa = 1.5: the moving ion and its micromotion blur the
//     threshold).  Polynomial form of b^4 < kappa^4 b_c^4:  |d x u|^4 mu < 8 kappa^4 C4 |u|^2.
// (2) Among them the slow ones take longest: the flight alone lasts ~1/u, and the complexes that
//     survive until t_max are low-energy ones (of the 12 longest trajectories of the bench
//     workload all have u^2 < <u^2>/2; measured).
// Three classes, queued in this order, each a stage of the schedule:
//     0: candidates with u^2 < <u^2>/2   1: the other candidates, and anything with u^2 < <u^2>/10
//     2: the rest
// so that the longest trajectories start their sequential run in the six-lane integrator after the
// first few per cent of the work instead of anywhere.  Affects scheduling only, never a result.
constexpr int kCntClass = 24;    // counters: trajectories per class (3)
constexpr int kCntCursor = 28;   // counters: placement cursors (3)
constexpr int kCntMeanU2 = 60;   // counters: <u^2> (double bits)

struct PlanArgs {
    double mu, c4k;  // reduced mass, 8 kappa^4 C4
    double slow0, slow1;  // class thresholds as fractions of <u^2>
};

__device__ __forceinline__ double rel_speed2(const double* __restrict__ y0, long long N, long long i)
{
    const double u0 = y0[9 * N + i] - y0[3 * N + i], u1 = y0[10 * N + i] - y0[4 * N + i],
                 u2 = y0[11 * N + i] - y0[5 * N + i];
    return u0 * u0 + u1 * u1 + u2 * u2;
}

__device__ __forceinline__ int plan_class(const double* __restrict__ y0, long long N, long long i, const PlanArgs& A,
                                          double mean_u2)
{
    const double d0 = y0[6 * N + i] - y0[0 * N + i], d1 = y0[7 * N + i] - y0[1 * N + i],
                 d2 = y0[8 * N + i] - y0[2 * N + i];
    const double u0 = y0[9 * N + i] - y0[3 * N + i], u1 = y0[10 * N + i] - y0[4 * N + i],
                 u2 = y0[11 * N + i] - y0[5 * N + i];
    const double c0 = d1 * u2 - d2 * u1, c1 = d2 * u0 - d0 * u2, c2 = d0 * u1 - d1 * u0;
    const double l2 = c0 * c0 + c1 * c1 + c2 * c2;
    const double usq = u0 * u0 + u1 * u1 + u2 * u2;
    const bool cand = (l2 * l2 * A.mu < A.c4k * usq);
    if (cand && usq < A.slow0 * mean_u2) return 0;
    if (cand || usq < A.slow1 * mean_u2) return 1;
    return 2;
}

// <u^2> over the first min(N, 65536) trajectories (a sample is enough for a scheduling threshold)
__global__ void __launch_bounds__(1024)
plan_mean_kernel(const double* __restrict__ y0, const long long N, unsigned long long* __restrict__ counters)
{
    __shared__ double part[32];
    const long long n = N < 65536 ? N : 65536;
    double s = 0.0;
    for (long long i = threadIdx.x; i < n; i += blockDim.x) s += rel_speed2(y0, N, i);
    for (int off = 16; off > 0; off >>= 1) s += __shfl_down_sync(0xffffffffu, s, off);
    if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x < 32) {
        s = (threadIdx.x < (blockDim.x >> 5)) ? part[threadIdx.x] : 0.0;
        for (int off = 16; off > 0; off >>= 1) s += __shfl_down_sync(0xffffffffu, s, off);
        if (threadIdx.x == 0) counters[kCntMeanU2] = (unsigned long long)__double_as_longlong(s / (double)n);
    }
}

// PLACE = 0: count the classes; PLACE = 1: write order[] (cursors set by plan_bounds_kernel)
template <int PLACE>
__global__ void __launch_bounds__(256)
plan_kernel(const double* __restrict__ y0, const long long N, const PlanArgs A, long long* __restrict__ order,
            unsigned long long* __restrict__ counters)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const unsigned FULL = 0xffffffffu;
    const double mean_u2 = __longlong_as_double((long long)counters[kCntMeanU2]);
    const int cls = (i < N) ? plan_class(y0, N, i, A, mean_u2) : -1;
    const int lane = threadIdx.x & 31;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const unsigned m = __ballot_sync(FULL, cls == c);
        if (m == 0u) continue;
        unsigned long long base = 0;
        if (lane == 0) base = atomicAdd(&counters[(PLACE ? kCntCursor : kCntClass) + c], (unsigned long long)__popc(m));
        if (PLACE) {
            base = __shfl_sync(FULL, base, 0);
            if (cls == c) order[base + __popc(m & ((1u << lane) - 1u))] = i;
        }
    }
}

// cursors at the class starts; bound[0..3] = the three stages' ranges of order[].  A stage is a
// class, except that empty classes at the end are skipped so that the LAST stage (the one whose
// six-lane pass has the whole GPU) is never empty while an earlier one is not: with a degenerate
// input (every trajectory in one class, e.g. a fixed launch speed) all the work is in the last stage.
__global__ void plan_bounds_kernel(unsigned long long* counters, int bound0, int front)
{
    unsigned long long start[4];
    unsigned long long acc = 0;
    for (int c = 0; c < 3; ++c) {
        start[c] = acc;
        counters[kCntCursor + c] = acc;
        acc += counters[kCntClass + c];
        if (c == 1) counters[front] = acc;  // classes 0 and 1 (diagnostics)
    }
    start[3] = acc;
    int last = 2;  // last non-empty class
    while (last > 0 && start[last + 1] == start[last]) --last;
    const int shift = 2 - last;  // stage s holds class s - shift (stages below `shift` are empty)
    for (int st = 0; st <= 3; ++st) {
        const int c = st - shift;
        counters[bound0 + st] = (c <= 0) ? 0 : start[c];
    }
    counters[bound0 + 3] = acc;
}

// without a plan: one stage over [0, N)
__global__ void bounds_kernel(unsigned long long* counters, int bound0, unsigned long long N)
{
    counters[bound0] = 0;
    counters[bound0 + 1] = N;
}

// Head start for the split pass of the previous stage: it is next in ITS stream's order and must take
// its SMs before the bulk pass of this stage (other stream) fills them; both become ready when the
// previous bulk pass ends.  Waits until the split pass has stamped its start (or at most `ns`).
__global__ void head_start_kernel(const unsigned long long* started, unsigned long long ns)
{
    const unsigned long long t0 = global_ns();
    while (*(volatile const unsigned long long*)started == 0ULL && global_ns() - t0 < ns) __nanosleep(500);
}

// counters[dst] = min(counters[src], cap): freezes the number of checkpoint slots written so far
__global__ void snapshot_kernel(unsigned long long* counters, int dst, int src, unsigned long long cap)
{
    const unsigned long long v = counters[src];
    counters[dst] = v < cap ? v : cap;
}

// ------------------------------------------------------------------------------------------
// test hook: one attempted step per thread
// ------------------------------------------------------------------------------------------
template <int TRAP>
__global__ void __launch_bounds__(kBlock)
step_once_kernel(const KParams P, const double* __restrict__ y, const double* __restrict__ t,
                 const double* __restrict__ h, const long long N, double* __restrict__ ynew,
                 double* __restrict__ err)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    Traj T;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        T.X[k] = y[(0 + k) * N + i];
        T.V[k] = y[(3 + k) * N + i];
        T.X[3 + k] = y[(6 + k) * N + i];
        T.V[3 + k] = y[(9 + k) * N + i];
    }
    T.c.t = t[i];
    T.c.h = h[i];
    T.c.flags = 0u;
    double r2;
    Attempt R;
    const double D[3] = {T.X[0] - T.X[3], T.X[1] - T.X[4], T.X[2] - T.X[5]};
    const double Xi[3] = {T.X[0], T.X[1], T.X[2]};
    // RF trap: the branch-free cos where it is valid, libdevice's beyond (the integrator makes
    // this choice once per call on the host, from t0 and t_max)
    if (trap_of(TRAP) == TRAP_RF && !(fabs(P.omega) * (fabs(T.c.t) + fabs(T.c.h)) < 0.99 * kCosMaxArg)) {
        constexpr int BIG = TRAP_RF_BIG + 4 * pot_of(TRAP);
        accel<BIG>(P, trap_cos<BIG>(P, T.c.t), D, Xi, T.A1, r2);
        dp45_attempt<BIG>(P, T, R);
    } else {
        accel<TRAP>(P, trap_cos<TRAP>(P, T.c.t), D, Xi, T.A1, r2);
        dp45_attempt<TRAP>(P, T, R);
    }
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        ynew[(0 + k) * N + i] = R.X[k];
        ynew[(3 + k) * N + i] = R.V[k];
        ynew[(6 + k) * N + i] = R.X[3 + k];
        ynew[(9 + k) * N + i] = R.V[3 + k];
    }
    err[i] = R.err;
}

// ------------------------------------------------------------------------------------------
// histogram
// ------------------------------------------------------------------------------------------
// number of edges <= v (0 = underflow, nb + 1 = overflow); NaN -> nb + 1
__device__ __forceinline__ int bin_of(const double* __restrict__ edges, int nb, double v)
{
    if (v != v) return nb + 1;
    int lo = 0, hi = nb + 1;  // count of edges[0..nb] that are <= v lies in [lo, hi]
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if (edges[mid] <= v)
            lo = mid + 1;
        else
            hi = mid;
    }
    return lo;
}

// warp-aggregated increment of a shared-memory bin: lanes that hit the same bin elect one
// leader that adds the group's population count (active lanes only).
__device__ __forceinline__ void agg_inc(unsigned int* bins, int bin)
{
    const unsigned act = __activemask();
    const unsigned grp = __match_any_sync(act, bin);
    if ((threadIdx.x & 31) == __ffs(grp) - 1) atomicAdd(&bins[bin], (unsigned)__popc(grp));
}

struct HistArgs {
    const double *angle, *lifetime;
    const int *n_acc, *n_rej, *n_turn, *status;
    const unsigned char* complex_flag;
    const double *angle_edges, *life_edges;
    int na, nl, nt;
    unsigned long long *h_angle, *h_life, *h_turn, *h_status, *h_totals;
};

__global__ void __launch_bounds__(256)
histogram_kernel(const HistArgs a, const long long N)
{
    extern __shared__ unsigned char smem_raw[];
    double* s_ae = reinterpret_cast<double*>(smem_raw);
    double* s_le = s_ae + (a.na + 1);
    unsigned int* s_angle = reinterpret_cast<unsigned int*>(s_le + (a.nl + 1));
    unsigned int* s_life = s_angle + (a.na + 2);
    unsigned int* s_turn = s_life + (a.nl + 2);
    unsigned int* s_status = s_turn + a.nt;
    const int nbins_total = (a.na + 2) + (a.nl + 2) + a.nt + 4;
    for (int i = threadIdx.x; i <= a.na; i += blockDim.x) s_ae[i] = a.angle_edges[i];
    for (int i = threadIdx.x; i <= a.nl; i += blockDim.x) s_le[i] = a.life_edges[i];
    for (int i = threadIdx.x; i < nbins_total; i += blockDim.x) s_angle[i] = 0u;
    __syncthreads();

    unsigned long long sum_acc = 0, sum_rej = 0, n_cplx = 0, n_traj = 0;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += stride) {
        agg_inc(s_angle, bin_of(s_ae, a.na, a.angle[i]));
        const bool cplx = a.complex_flag[i] != 0;
        if (cplx) agg_inc(s_life, bin_of(s_le, a.nl, a.lifetime[i]));
        const int nt = a.n_turn[i];
        agg_inc(s_turn, nt < 0 ? 0 : (nt >= a.nt ? a.nt - 1 : nt));
        agg_inc(s_status, a.status[i] & 3);
        sum_acc += (unsigned long long)a.n_acc[i];
        sum_rej += (unsigned long long)a.n_rej[i];
        n_cplx += cplx ? 1u : 0u;
        n_traj += 1u;
    }
    // totals: warp shuffle reduction, one global atomic per warp and quantity
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        sum_acc += __shfl_down_sync(0xffffffffu, sum_acc, off);
        sum_rej += __shfl_down_sync(0xffffffffu, sum_rej, off);
        n_cplx += __shfl_down_sync(0xffffffffu, n_cplx, off);
        n_traj += __shfl_down_sync(0xffffffffu, n_traj, off);
    }
    if ((threadIdx.x & 31) == 0) {
        if (sum_acc) atomicAdd(&a.h_totals[0], sum_acc);
        if (sum_rej) atomicAdd(&a.h_totals[1], sum_rej);
        if (n_cplx) atomicAdd(&a.h_totals[2], n_cplx);
        if (n_traj) atomicAdd(&a.h_totals[3], n_traj);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < a.na + 2; i += blockDim.x)
        if (s_angle[i]) atomicAdd(&a.h_angle[i], (unsigned long long)s_angle[i]);
    for (int i = threadIdx.x; i < a.nl + 2; i += blockDim.x)
        if (s_life[i]) atomicAdd(&a.h_life[i], (unsigned long long)s_life[i]);
    for (int i = threadIdx.x; i < a.nt; i += blockDim.x)
        if (s_turn[i]) atomicAdd(&a.h_turn[i], (unsigned long long)s_turn[i]);
    for (int i = threadIdx.x; i < 4; i += blockDim.x)
        if (s_status[i]) atomicAdd(&a.h_status[i], (unsigned long long)s_status[i]);
}

// ------------------------------------------------------------------------------------------
// NEXT-3: replay of one trajectory with every accepted step recorded
// ------------------------------------------------------------------------------------------
// One thread, the same functions as integrate_kernel: the replay is bit-identical to what
// aig_integrate computed for these initial conditions (the paper recomputes its longest-lived
// trajectory "with the same exact initial conditions" and gets different bounces, :509).
template <int TRAP>
__global__ void __launch_bounds__(32)
trace_kernel(const KParams P, const double* __restrict__ y0, const long long cap, double* __restrict__ t_out,
             double* __restrict__ y_out, long long* __restrict__ n_out)
{
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    Traj T;
    ColdRegs C;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        T.X[k] = y0[0 + k];
        T.V[k] = y0[3 + k];
        T.X[3 + k] = y0[6 + k];
        T.V[3 + k] = y0[9 + k];
    }
    init_traj<TRAP>(P, T, C);
    int st = -1;
    while (st < 0) {
        const int before = T.c.n_acc;
        Attempt R;
        dp45_attempt<TRAP>(P, T, R);
        bool first_turn;
        st = finish_attempt(P, T, C, R, first_turn);
        if (T.c.n_acc != before) {
            const long long j = (long long)before;
            if (j < cap) {
                t_out[j] = T.c.t;
#pragma unroll
                for (int k = 0; k < 3; ++k) {
                    y_out[(0 + k) * cap + j] = T.X[k];
                    y_out[(3 + k) * cap + j] = T.V[k];
                    y_out[(6 + k) * cap + j] = T.X[3 + k];
                    y_out[(9 + k) * cap + j] = T.V[3 + k];
                }
            }
        }
    }
    n_out[0] = T.c.n_acc;
    n_out[1] = st;
    n_out[2] = C.n_rej();
    n_out[3] = C.n_turn();
}

// ------------------------------------------------------------------------------------------
// NEXT-1: the paper's remaining observables and its outliers (:521)
// ------------------------------------------------------------------------------------------
// HBM-bound: reads the final state (96 B) and the initial atom velocity (24 B), writes 24 B; with
// `position` 24 B more are read (the ion position at the first bounce) and 8 B more written.
__global__ void __launch_bounds__(256)
observables_kernel(const double* __restrict__ y0, const double* __restrict__ yf, const long long N,
                   const double m_ion, const double m_atom, double* __restrict__ dist, double* __restrict__ ke,
                   double* __restrict__ transfer, const double* __restrict__ x_turn1, double* __restrict__ position)
{
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += stride) {
        const double d0 = yf[6 * N + i] - yf[0 * N + i], d1 = yf[7 * N + i] - yf[1 * N + i],
                     d2 = yf[8 * N + i] - yf[2 * N + i];
        const double v0 = yf[3 * N + i], v1 = yf[4 * N + i], v2 = yf[5 * N + i];
        const double w0 = yf[9 * N + i] - y0[9 * N + i], w1 = yf[10 * N + i] - y0[10 * N + i],
                     w2 = yf[11 * N + i] - y0[11 * N + i];
        dist[i] = sqrt(sum3(d0 * d0, d1 * d1, d2 * d2));
        ke[i] = (0.5 * m_ion) * sum3(v0 * v0, v1 * v1, v2 * v2);
        transfer[i] = m_atom * sqrt(sum3(w0 * w0, w1 * w1, w2 * w2));
        if (position) {  // NaN where there was no bounce (x_turn1 holds NaN there)
            const double p0 = x_turn1[0 * N + i], p1 = x_turn1[1 * N + i], p2 = x_turn1[2 * N + i];
            position[i] = sqrt(sum3(p0 * p0, p1 * p1, p2 * p2));
        }
    }
}

// arg-min / arg-max of eight observables in one pass: (value, index) pairs, the smaller index wins
// a tie, NaNs are skipped, index -1 = nothing seen.
constexpr int kOutlierObs = 8;  // angle, n_turn, lifetime, transfer, dist, n_acc, KE, position
struct Extreme {
    double v;
    long long i;
};
__device__ __forceinline__ Extreme pick_min(const Extreme a, const Extreme b)
{
    const bool tb = (b.i >= 0) && ((a.i < 0) || (b.v < a.v) || ((b.v == a.v) && (b.i < a.i)));
    return tb ? b : a;
}
__device__ __forceinline__ Extreme pick_max(const Extreme a, const Extreme b)
{
    const bool tb = (b.i >= 0) && ((a.i < 0) || (b.v > a.v) || ((b.v == a.v) && (b.i < a.i)));
    return tb ? b : a;
}
__device__ __forceinline__ Extreme shfl_extreme(const Extreme e, int off)
{
    Extreme r;
    r.v = __shfl_down_sync(0xffffffffu, e.v, off);
    r.i = __shfl_down_sync(0xffffffffu, e.i, off);
    return r;
}

struct OutlierArgs {
    const double *angle, *lifetime, *transfer, *dist, *ke;
    const double* position;        // may be nullptr: the row then reads -1, -1
    const int *n_turn, *n_acc;
    Extreme* partial;              // [gridDim.x][kOutlierObs][2]
    unsigned int* ticket;          // blocks that have finished
    long long* result;             // [kOutlierObs][2]: index of the minimum, of the maximum
};

// the eight observables of trajectory i as doubles (a missing position array reads NaN: skipped)
__device__ __forceinline__ void outlier_load(const OutlierArgs& a, long long i, double (&x)[kOutlierObs])
{
    x[0] = a.angle[i];
    x[1] = (double)a.n_turn[i];
    x[2] = a.lifetime[i];
    x[3] = a.transfer[i];
    x[4] = a.dist[i];
    x[5] = (double)a.n_acc[i];
    x[6] = a.ke[i];
    x[7] = a.position ? a.position[i] : nan("");
}
// a thread visits its indices in ascending order, so a strict comparison keeps the smallest index of a
// tie; the running extrema carry the visit number (32 bits; -1 = nothing yet), not the index
struct Running {
    double v;
    int n;
};
__device__ __forceinline__ void outlier_fold(const double (&x)[kOutlierObs], int n, Running (&lo)[kOutlierObs],
                                             Running (&hi)[kOutlierObs])
{
#pragma unroll
    for (int k = 0; k < kOutlierObs; ++k) {
        const bool ok = (x[k] == x[k]);
        const bool tl = ok & ((x[k] < lo[k].v) | (lo[k].n < 0));
        const bool th = ok & ((x[k] > hi[k].v) | (hi[k].n < 0));
        lo[k].v = tl ? x[k] : lo[k].v;
        lo[k].n = tl ? n : lo[k].n;
        hi[k].v = th ? x[k] : hi[k].v;
        hi[k].n = th ? n : hi[k].n;
    }
}

__global__ void __launch_bounds__(256, 2)
outliers_kernel(const OutlierArgs a, const long long N)
{
    __shared__ Extreme s_part[8][kOutlierObs][2];
    __shared__ bool s_last;
    Running rlo[kOutlierObs], rhi[kOutlierObs];
#pragma unroll
    for (int k = 0; k < kOutlierObs; ++k) {
        rlo[k].v = rhi[k].v = 0.0;
        rlo[k].n = rhi[k].n = -1;
    }
    // two trajectories per iteration, all sixteen loads issued before the first comparison (HBM latency)
    const long long stride = (long long)gridDim.x * blockDim.x;
    const long long start = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    long long i = start;
    int n = 0;  // visit number: index = start + n * stride
    for (; i + stride < N; i += 2 * stride, n += 2) {
        double x0[kOutlierObs], x1[kOutlierObs];
        outlier_load(a, i, x0);
        outlier_load(a, i + stride, x1);
        outlier_fold(x0, n, rlo, rhi);
        outlier_fold(x1, n + 1, rlo, rhi);
    }
    if (i < N) {
        double x0[kOutlierObs];
        outlier_load(a, i, x0);
        outlier_fold(x0, n, rlo, rhi);
    }
    Extreme lo[kOutlierObs], hi[kOutlierObs];
#pragma unroll
    for (int k = 0; k < kOutlierObs; ++k) {
        lo[k].v = rlo[k].v;
        lo[k].i = rlo[k].n < 0 ? -1 : start + (long long)rlo[k].n * stride;
        hi[k].v = rhi[k].v;
        hi[k].i = rhi[k].n < 0 ? -1 : start + (long long)rhi[k].n * stride;
    }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int k = 0; k < kOutlierObs; ++k) {
        for (int off = 16; off > 0; off >>= 1) {
            lo[k] = pick_min(lo[k], shfl_extreme(lo[k], off));
            hi[k] = pick_max(hi[k], shfl_extreme(hi[k], off));
        }
        if (lane == 0) {
            s_part[warp][k][0] = lo[k];
            s_part[warp][k][1] = hi[k];
        }
    }
    __syncthreads();
    if (threadIdx.x < kOutlierObs * 2) {
        const int k = threadIdx.x >> 1, m = threadIdx.x & 1;
        Extreme e = s_part[0][k][m];
        for (int w = 1; w < (int)(blockDim.x >> 5); ++w) e = m ? pick_max(e, s_part[w][k][m]) : pick_min(e, s_part[w][k][m]);
        a.partial[((size_t)blockIdx.x * kOutlierObs + k) * 2 + m] = e;
    }
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) s_last = (atomicAdd(a.ticket, 1u) == gridDim.x - 1);
    __syncthreads();
    if (s_last) {
        // the last block to finish folds the partials: 16 threads per (observable, min | max); the order
        // of the fold does not matter ((value, index) pairs are totally ordered)
        __threadfence();
        const int c = threadIdx.x >> 4, sub = threadIdx.x & 15;
        const bool act = c < kOutlierObs * 2;
        const int k = act ? (c >> 1) : 0, m = c & 1;
        Extreme e{0.0, -1};
        if (act)
#pragma unroll 4
            for (unsigned b = sub; b < gridDim.x; b += 16) {
                const Extreme f = a.partial[((size_t)b * kOutlierObs + k) * 2 + m];
                e = m ? pick_max(e, f) : pick_min(e, f);
            }
        for (int off = 8; off > 0; off >>= 1) {
            const Extreme f = shfl_extreme(e, off);
            e = m ? pick_max(e, f) : pick_min(e, f);
        }
        if (act && sub == 0) a.result[k * 2 + m] = e.i;
    }
}

// ------------------------------------------------------------------------------------------
// FP64 roofline probe: ILP independent FMA chains per thread, all in registers
// ------------------------------------------------------------------------------------------
template <int ILP>
__global__ void __launch_bounds__(256)
dfma_probe_kernel(double* out, int iters, double a, double b)
{
    double x[ILP];
#pragma unroll
    for (int j = 0; j < ILP; ++j) x[j] = 1.0 + 1e-3 * (threadIdx.x + j);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int rep = 0; rep < 8; ++rep) {
#pragma unroll
            for (int j = 0; j < ILP; ++j) x[j] = fma(x[j], a, b);
        }
    }
    double s = 0.0;
#pragma unroll
    for (int j = 0; j < ILP; ++j) s += x[j];
    if (s == 123.456) out[0] = s;  // keeps the chains alive, never true in practice
}

}  // namespace aig

// ==========================================================================================
// host side: C ABI
// ==========================================================================================
using namespace aig;

namespace {

std::atomic<unsigned long long> g_kernel_launches{0};  // aig_kernel_launches()

bool finite(double x) { return std::isfinite(x); }

int check_params(const aig_params* p, double t_max, double rtol, double atol)
{
    if (!p) return AIG_ERR_NULL;
    if (!(rtol > 0.0) || !(atol >= 0.0) || !finite(rtol) || !finite(atol)) return AIG_ERR_TOL;
    if (!finite(t_max) || !finite(p->t0) || !(t_max > p->t0)) return AIG_ERR_TIME;
    if (!(p->m_ion > 0.0) || !(p->m_atom > 0.0) || !finite(p->m_ion) || !finite(p->m_atom))
        return AIG_ERR_PARAM;
    if (!finite(p->C4) || !finite(p->C8) || !finite(p->omega_rf)) return AIG_ERR_PARAM;
    for (int k = 0; k < 3; ++k)
        if (!finite(p->a[k]) || !finite(p->q[k])) return AIG_ERR_PARAM;
    if (p->max_steps < 1) return AIG_ERR_PARAM;
    if (!(p->n_att == 0 && p->n_rep == 0) && !(p->n_att >= 1 && p->n_att < p->n_rep && p->n_rep <= 32)) return AIG_ERR_PARAM;
    if (std::isnan(p->r_exit) || std::isnan(p->r_turn)) return AIG_ERR_PARAM;
    return AIG_OK;
}

int trap_mode(const aig_params* p, double t_max)
{
    const double w2 = p->omega_rf * p->omega_rf;
    bool any_a = false, any_q = false;
    for (int k = 0; k < 3; ++k) {
        any_a = any_a || (p->a[k] * w2 != 0.0);
        any_q = any_q || (p->q[k] * w2 != 0.0);
    }
    if (!any_q) return any_a ? TRAP_STATIC : TRAP_NONE;
    // the branch-free cos is valid for |Omega t| < kCosMaxArg; beyond that use libdevice's cos
    const double phase = std::fabs(p->omega_rf) * std::fmax(std::fabs(p->t0), std::fabs(t_max));
    return (phase < 0.99 * kCosMaxArg) ? TRAP_RF : TRAP_RF_BIG;
}

// potential kind: 0, 0 (or 4, 8) = the benchmark potential's fast path, anything else the general one
bool general_potential(const aig_params* p)
{
    return !((p->n_att == 0 && p->n_rep == 0) || (p->n_att == 4 && p->n_rep == 8));
}

KParams make_kparams(const aig_params* p, double t_max, double rtol, double atol)
{
    KParams K;
    const int n = p->n_att ? p->n_att : 4, m = p->n_rep ? p->n_rep : 8;
    K.g4i = -(double)n * p->C4 / p->m_ion;
    K.g8i = (double)m * p->C8 / p->m_ion;
    K.g4a = (double)n * p->C4 / p->m_atom;
    K.g8a = -(double)m * p->C8 / p->m_atom;
    K.pot_sqrt = ((n | m) & 1) ? 1 : 0;
    K.pot_e_att = K.pot_sqrt ? n + 2 : (n + 2) / 2;
    K.pot_e_rep = K.pot_sqrt ? m + 2 : (m + 2) / 2;
    const double w2 = p->omega_rf * p->omega_rf;
    for (int k = 0; k < 3; ++k) {
        K.wa[k] = p->a[k] * w2 / 4.0;
        K.wb[k] = p->q[k] * w2 / 2.0;
    }
    K.omega = p->omega_rf;
    K.half_omega = 0.5 * p->omega_rf;
    K.t0 = p->t0;
    K.t_max = t_max;
    K.hmax = 0.1 * (t_max - p->t0);
    K.rtol = rtol;
    K.inv_rtol = 1.0 / rtol;
    K.thr = atol / rtol;
    K.rho_scale = 1.0 / (0.8 * std::pow(rtol, 0.2));
    K.r_exit2 = (p->r_exit > 0.0) ? p->r_exit * p->r_exit : INFINITY;
    K.r_turn2 = p->r_turn * p->r_turn;  // +inf stays +inf
    if (p->r_turn < 0.0) K.r_turn2 = 0.0;
    K.max_steps = p->max_steps;
    return K;
}

bool aligned(const void* ptr, size_t a) { return (reinterpret_cast<uintptr_t>(ptr) % a) == 0; }

// ---- schedule of one aig_integrate call ------------------------------------------------------
//   plan        order[] in three classes (plan_*_kernel), bound[] = where each class starts
//   stage i     (i = 0, 1, 2 = class; each on its own stream, stage 0 on the caller's):
//     bulk i    per-thread integrator over class i; what outlives `budget` accepted steps, or is
//               still running `tail_iters` iterations after the queue ran dry, is suspended into
//               the next free checkpoint slots
//     split i   six-lane integrator over the slots bulk i wrote.  Stage i + 1 starts when bulk i is
//               complete (event), so split i runs BESIDE bulk i + 1: the longest trajectories
//               (10^2..10^3 x the mean number of steps, nearly all in class 0) start their long
//               sequential run after a few per cent of the work.  Beside a bulk pass it takes
//               `split_sms` SMs for itself (one 8-warp block per SM that asks for the whole shared
//               memory, so that no bulk block can share its FP64 pipes); that bulk pass is sized
//               for the remaining SMs and lets the split pass take its SMs first (head_start_kernel).
//   join        the caller's stream waits for the side streams.
// No kernel waits for another one's progress (no polling for work): every dependency is a stream
// order or an event; head_start_kernel only delays a launch, by at most 200 us.
// Checkpoint slots: min(N, max(2^20, N/4)).  Hand-overs are bounded by 3 stages x (soft_cap + resident lanes)
// ~ 1.6e5, so the capacity test in the kernel is a safety net, not a working regime.
constexpr long long kMinSlots = 1 << 20;

struct SchedConfig {
    int tail_iters = 256;     // iterations a warp keeps stepping after the queue ran dry
    int budget = 2048;        // accepted steps after which the per-thread integrator hands a trajectory over
    int split_sms = 32;       // SMs a six-lane pass takes for itself beside a bulk pass (one 8-warp block each)
    int split_grid_b = 8;     // last six-lane pass: one-warp blocks per SM (it has the GPU to itself)
    int soft_cap = 16384;     // budget hand-overs per bulk stage (drain hand-overs come on top)
    int mean_factor = 4;      // ... and only of trajectories this many times longer than the finished ones' mean
    int drain_lanes = 10;     // queue empty: a warp hands over what it still runs once this few lanes are alive
    double slow0 = 0.5;       // class 0: candidates with u^2 < slow0 <u^2>
    double slow1 = 0.1;       // class 1 also takes anything with u^2 < slow1 <u^2>
    int refill_batch = 8;     // idle lanes of a warp that trigger its refill ...
    int refill_wait = 16;     // ... or iterations one of them has waited
    int plan = 1;             // 0: natural order, one bulk launch
    double kappa = 1.5;       // candidates: b < kappa * Langevin radius
};

std::mutex g_sched_mutex;
SchedConfig g_sched;          // guarded by g_sched_mutex
bool g_sched_init = false;

// the schedule in force: defaults, overridden once by AIG_SCHED="tail_iters,budget,split_sms,
// split_grid_b,plan,kappa" (tuning aid) and at any time by aig_set_schedule()
SchedConfig sched_config()
{
    std::lock_guard<std::mutex> lock(g_sched_mutex);
    if (!g_sched_init) {
        SchedConfig c;
        if (const char* e = std::getenv("AIG_SCHED")) {
            int a = c.tail_iters, b = c.budget, ga = c.split_sms, gb = c.split_grid_b, pl = c.plan;
            double kp = c.kappa;
            const int got = std::sscanf(e, "%d,%d,%d,%d,%d,%lf", &a, &b, &ga, &gb, &pl, &kp);
            if (got >= 1 && a >= 0) c.tail_iters = a;
            if (got >= 2 && b >= 1) c.budget = b;
            if (got >= 3 && ga >= 1) c.split_sms = ga;
            if (got >= 4 && gb >= 1) c.split_grid_b = gb;
            if (got >= 5) c.plan = pl;
            if (got >= 6 && kp >= 0.0) c.kappa = kp;
        }
        if (const char* e = std::getenv("AIG_REFILL")) {  // "batch,wait,slow0,slow1,mean_factor,drain_lanes" (tuning aid)
            int b = c.refill_batch, w = c.refill_wait, mf = c.mean_factor, dl = c.drain_lanes;
            double s0 = c.slow0, s1 = c.slow1;
            const int got = std::sscanf(e, "%d,%d,%lf,%lf,%d,%d", &b, &w, &s0, &s1, &mf, &dl);
            if (got >= 5 && mf >= 0) c.mean_factor = mf;
            if (got >= 6 && dl >= 0) c.drain_lanes = dl;
            if (got >= 1 && b >= 1) c.refill_batch = b;
            if (got >= 2 && w >= 0) c.refill_wait = w;
            if (got >= 3 && s0 >= 0.0) c.slow0 = s0;
            if (got >= 4 && s1 >= 0.0) c.slow1 = s1;
        }
        g_sched = c;
        g_sched_init = true;
    }
    return g_sched;
}

long long slot_capacity(long long N) { return std::min(N < 1 ? 1 : N, std::max(kMinSlots, N / 4)); }

size_t round_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// workspace: 64 uint64 counters | order[N] (int64) | checkpoint slots
constexpr size_t kCounterBytes = 64 * sizeof(unsigned long long);
size_t order_bytes(long long N) { return round_up((size_t)(N < 1 ? 1 : N) * sizeof(long long), 256); }
size_t ckpt_buffer_bytes(long long cap) { return round_up((size_t)cap * kCkptBytesPerSlot, 256); }

// counters (uint64 each).  Stage i of the schedule: bulk pass over order[bound[i], bound[i+1]), its
// hand-overs are the slots [snap[i], snap[i+1]).
constexpr int kMaxStages = 4;
enum Counter {
    kCntFront = 0,   // plan: candidates placed (= n_front)
    kCntZero = 2,    // constant 0
    kCntN = 3,       // constant N
    kCntSlots = 4,   // checkpoint slots handed out so far (may overshoot the capacity)
    kCntBound = 5,   // bound[0 .. kMaxStages]
    kCntSnap = 10,   // snap[0 .. kMaxStages], snap[0] = 0
    kCntQueueBulk = 16,   // work queue of bulk pass i
    kCntQueueSplit = 20,  // work queue of split pass i
    kCntLoaded = 61,      // diagnostics: trajectories split pass i has taken (its own and earlier stages')
    kCntStats = 52        // [2 i], [2 i + 1]: accepted steps / number of the trajectories bulk pass i has finished
};

Ckpt ckpt_at(unsigned char* base, long long cap)
{
    Ckpt c;
    c.d = reinterpret_cast<double*>(base);
    c.idx = reinterpret_cast<long long*>(base + (size_t)cap * kCkptDoubles * 8);
    c.i = reinterpret_cast<int*>(base + (size_t)cap * (kCkptDoubles * 8 + 8));
    c.cap = cap;
    return c;
}

template <int TRAP>
int bulk_capacity(int* blocks_per_sm, int* sm_count)
{
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return AIG_ERR_CUDA;
    if (cudaDeviceGetAttribute(sm_count, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
        return AIG_ERR_CUDA;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(blocks_per_sm, integrate_kernel<TRAP, kBlock, kBlocksPerSM>,
                                                      kBlock, 0) != cudaSuccess)
        return AIG_ERR_CUDA;
    if (*blocks_per_sm < 1) return AIG_ERR_CUDA;
    return AIG_OK;
}

// side streams (stage i >= 1 runs on stream i - 1) and the events that chain and join them, one set
// per device
struct SideStreams {
    cudaStream_t stream[kMaxStages - 1] = {};
    cudaEvent_t done[kMaxStages] = {};   // done[i]: bulk pass i and its snapshot are complete
    cudaEvent_t join[kMaxStages - 1] = {};
    bool ok = false;
};
std::mutex g_side_mutex;

SideStreams* side_streams()
{
    static SideStreams side[64];
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return nullptr;
    std::lock_guard<std::mutex> lock(g_side_mutex);
    SideStreams& s = side[dev];
    if (!s.ok) {
        int lo = 0, hi = 0;
        if (cudaDeviceGetStreamPriorityRange(&lo, &hi) != cudaSuccess) return nullptr;
        for (int i = 0; i < kMaxStages - 1; ++i) {
            if (cudaStreamCreateWithPriority(&s.stream[i], cudaStreamNonBlocking, lo) != cudaSuccess) return nullptr;
            if (cudaEventCreateWithFlags(&s.join[i], cudaEventDisableTiming) != cudaSuccess) return nullptr;
        }
        for (int i = 0; i < kMaxStages; ++i)
            if (cudaEventCreateWithFlags(&s.done[i], cudaEventDisableTiming) != cudaSuccess) return nullptr;
        s.ok = true;
    }
    return &s;
}

constexpr int kSplitMinBlocks = 8;  // register cap of the split kernel: 65536 / (8 x 32) = 256
#ifndef AIG_SPLIT_WARPS
#define AIG_SPLIT_WARPS 8
#endif
constexpr int kSplitWarps = AIG_SPLIT_WARPS;  // warps per block of the SM-owning variant: two per scheduler (a warp issues 30 % of the
                                              // time, so two barely slow each other while the queue is long; at the end each is alone)

template <int TRAP>
int launch_integrate(const aig_params* p, const KParams& K, const double* y0, long long N, const OutPtrs& O,
                     void* workspace, cudaStream_t st)
{
    const SchedConfig cfg = sched_config();
    const long long cap = slot_capacity(N);
    unsigned long long* counters = static_cast<unsigned long long*>(workspace);
    long long* order = reinterpret_cast<long long*>(static_cast<unsigned char*>(workspace) + kCounterBytes);
    const Ckpt slots = ckpt_at(static_cast<unsigned char*>(workspace) + kCounterBytes + order_bytes(N), cap);
    if (cudaMemsetAsync(counters, 0, kCounterBytes, st) != cudaSuccess) return AIG_ERR_CUDA;
    const unsigned long long n64 = (unsigned long long)N;
    if (cudaMemcpyAsync(counters + kCntN, &n64, sizeof(n64), cudaMemcpyHostToDevice, st) != cudaSuccess)
        return AIG_ERR_CUDA;

    {
        // CUDA loads a kernel's code at its first launch (lazy module loading), and loading may have to
        // wait for the kernels that are running: the first call would serialise the passes that are meant
        // to overlap.  Touch every kernel of the schedule before anything is enqueued.
        cudaFuncAttributes fa;
        if (cudaFuncGetAttributes(&fa, integrate_kernel<TRAP, kBlock, kBlocksPerSM>) != cudaSuccess ||
            cudaFuncGetAttributes(&fa, integrate_split_kernel<TRAP, kSplitWarps, 1>) != cudaSuccess ||
            cudaFuncGetAttributes(&fa, integrate_split_kernel<TRAP, 1, kSplitMinBlocks>) != cudaSuccess ||
            cudaFuncGetAttributes(&fa, plan_mean_kernel) != cudaSuccess ||
            cudaFuncGetAttributes(&fa, plan_kernel<0>) != cudaSuccess ||
            cudaFuncGetAttributes(&fa, plan_kernel<1>) != cudaSuccess ||
            cudaFuncGetAttributes(&fa, plan_bounds_kernel) != cudaSuccess ||
            cudaFuncGetAttributes(&fa, bounds_kernel) != cudaSuccess ||
            cudaFuncGetAttributes(&fa, snapshot_kernel) != cudaSuccess ||
            cudaFuncGetAttributes(&fa, head_start_kernel) != cudaSuccess)
            return AIG_ERR_CUDA;
    }
    int bps = 0, sms = 0;
    int rc = bulk_capacity<TRAP>(&bps, &sms);
    if (rc) return rc;
    const long long blocks = std::min((long long)bps * sms, (N + kBlock - 1) / kBlock);
    const bool plan = cfg.plan != 0 && p->C4 > 0.0 && (p->n_att == 0 || p->n_att == 4);  // the Langevin test is the r^-4 tail's
    // stages: the three classes of the plan; without a plan one stage over [0, N)
    const int stages = plan ? 3 : 1;
    SideStreams* side = stages > 1 ? side_streams() : nullptr;
    if (stages > 1 && !side) return AIG_ERR_CUDA;

    long long* order_arg = nullptr;
    if (plan) {
        PlanArgs A;
        A.mu = p->m_ion * p->m_atom / (p->m_ion + p->m_atom);
        const double k2 = cfg.kappa * cfg.kappa;
        A.c4k = 8.0 * k2 * k2 * p->C4;
        A.slow0 = cfg.slow0;
        A.slow1 = cfg.slow1;
        const unsigned pg = (unsigned)((N + 255) / 256);
        plan_mean_kernel<<<1, 1024, 0, st>>>(y0, N, counters);
        plan_kernel<0><<<pg, 256, 0, st>>>(y0, N, A, order, counters);
        plan_bounds_kernel<<<1, 1, 0, st>>>(counters, kCntBound, kCntFront);
        plan_kernel<1><<<pg, 256, 0, st>>>(y0, N, A, order, counters);
        g_kernel_launches += 4;
        order_arg = order;
    } else {
        bounds_kernel<<<1, 1, 0, st>>>(counters, kCntBound, (unsigned long long)N);
        g_kernel_launches++;
    }

    int dev = 0, smem_optin = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev) != cudaSuccess)
        return AIG_ERR_CUDA;
    if (cudaFuncSetAttribute(integrate_split_kernel<TRAP, kSplitWarps, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             smem_optin) != cudaSuccess)
        return AIG_ERR_CUDA;
    const long long own = std::max<long long>(1, std::min<long long>(cfg.split_sms, sms / 2));
    const long long blocks_beside = std::max<long long>(1, std::min<long long>(blocks, (long long)bps * (sms - own)));
    const unsigned split_last =
        (unsigned)std::min<long long>((long long)cfg.split_grid_b * sms, (cap + kGroupsPerWarp - 1) / kGroupsPerWarp);

    // Stage i on its own stream (stage 0: the caller's): bulk pass i, snapshot, [event done_i], split pass i.
    // Stage i + 1 waits for done_i, so bulk pass i + 1 runs beside split pass i; the split pass comes first
    // in its own stream's order and takes its SMs before the next bulk pass (other stream, event) arrives.
    for (int i = 0; i < stages; ++i) {
        cudaStream_t cs = (i == 0) ? st : side->stream[i - 1];
        if (i > 0) {
            if (cudaStreamWaitEvent(cs, side->done[i - 1], 0) != cudaSuccess) return AIG_ERR_CUDA;
            // split pass i - 1 stamps counters[kCntTime + 2 (2 + 2 (i - 1))] when its first block starts
            head_start_kernel<<<1, 1, 0, cs>>>(counters + kCntTime + 2 * (2 + 2 * (i - 1)), 200000ULL);
            g_kernel_launches++;
        }
        Sched S;
        S.order = order_arg;
        S.queue = counters + kCntQueueBulk + i;
        S.begin = counters + kCntBound + i;
        S.end = counters + kCntBound + i + 1;
        S.n_out = counters + kCntSlots;
        S.soft_base = counters + kCntSnap + i;
        S.soft_cap = cfg.soft_cap;
        S.out = slots;
        S.budget = cfg.budget;
        S.tail_iters = cfg.tail_iters;
        S.refill_batch = cfg.refill_batch;
        S.refill_wait = cfg.refill_wait;
        S.drain_lanes = cfg.drain_lanes;
        S.stats = counters + kCntStats + 2 * i;
        S.mean_factor = cfg.mean_factor;
        S.timeline = counters + kCntTime + 2 * (1 + 2 * i);
        const long long grid = (i == 0) ? blocks : blocks_beside;
        integrate_kernel<TRAP, kBlock, kBlocksPerSM><<<(unsigned)grid, kBlock, 0, cs>>>(K, y0, N, O, S);
        snapshot_kernel<<<1, 1, 0, cs>>>(counters, kCntSnap + i + 1, kCntSlots, (unsigned long long)cap);
        g_kernel_launches += 2;
        if (i + 1 < stages && cudaEventRecord(side->done[i], cs) != cudaSuccess) return AIG_ERR_CUDA;
        SplitSched T;
        T.in = slots;
        T.timeline = counters + kCntTime + 2 * (2 + 2 * i);
        T.loaded = counters + kCntLoaded + i;
        T.nq = i + 1;
        for (int j = 0; j <= i; ++j) {  // own range first, then the earlier stages'
            T.queue[j] = counters + kCntQueueSplit + (i - j);
            T.begin[j] = counters + kCntSnap + (i - j);
            T.end[j] = counters + kCntSnap + (i - j) + 1;
        }
        if (i + 1 < stages) {
            // beside the next bulk pass: one block per SM it owns (the dynamic shared memory request
            // leaves no room for a bulk block next to it)
            integrate_split_kernel<TRAP, kSplitWarps, 1><<<(unsigned)own, 32 * kSplitWarps, (size_t)smem_optin, cs>>>(K, y0, N, O, T);
        } else {
            integrate_split_kernel<TRAP, 1, kSplitMinBlocks><<<split_last, 32, 0, cs>>>(K, y0, N, O, T);
        }
        g_kernel_launches++;
        if (i > 0 && cudaEventRecord(side->join[i - 1], cs) != cudaSuccess) return AIG_ERR_CUDA;
    }
    for (int i = 1; i < stages; ++i)
        if (cudaStreamWaitEvent(st, side->join[i - 1], 0) != cudaSuccess) return AIG_ERR_CUDA;
    return cudaGetLastError() == cudaSuccess ? AIG_OK : AIG_ERR_CUDA;
}

}  // namespace

extern "C" {

int aig_version(void) { return AIG_VERSION; }

uint64_t aig_kernel_launches(void) { return g_kernel_launches.load(); }

int aig_set_schedule(int tail_iters, int budget, int split_sms, int split_grid, int plan, double kappa)
{
    if (tail_iters < 0 || budget < 1 || split_sms < 1 || split_grid < 1 || !(kappa >= 0.0)) return AIG_ERR_PARAM;
    (void)sched_config();  // settle the defaults / environment first
    std::lock_guard<std::mutex> lock(g_sched_mutex);
    g_sched.tail_iters = tail_iters;
    g_sched.budget = budget;
    g_sched.split_sms = split_sms;
    g_sched.split_grid_b = split_grid;
    g_sched.plan = plan;
    g_sched.kappa = kappa;
    return AIG_OK;
}

const char* aig_strerror(int code)
{
    switch (code) {
        case AIG_OK: return "ok";
        case AIG_ERR_NULL: return "required pointer is NULL";
        case AIG_ERR_SIZE: return "invalid size (N < 0, N too large, or bad bin count)";
        case AIG_ERR_TOL: return "invalid tolerance (rtol <= 0 or atol < 0)";
        case AIG_ERR_TIME: return "invalid time span (t_max <= t0)";
        case AIG_ERR_PARAM: return "invalid physical parameter";
        case AIG_ERR_ALIGN: return "misaligned device pointer";
        case AIG_ERR_CUDA: return "CUDA runtime error (no device, launch failure or out of memory)";
        default: return "unknown error code";
    }
}

size_t aig_workspace_bytes(int64_t N)
{
    // counters + work-queue order (8 B per trajectory) + checkpoint slots for suspended trajectories
    return kCounterBytes + order_bytes(N) + ckpt_buffer_bytes(slot_capacity(N));
}

int aig_integrate(const aig_params* p, const double* y0, int64_t N, double t_max, double rtol,
                  double atol, const aig_out* out, void* workspace, void* cuda_stream)
{
    int rc = check_params(p, t_max, rtol, atol);
    if (rc) return rc;
    if (N < 0 || N > (1LL << 40)) return AIG_ERR_SIZE;
    if (N == 0) return AIG_OK;
    if (!y0 || !out || !workspace) return AIG_ERR_NULL;
    if (!out->y_final || !out->t_final || !out->lifetime || !out->angle || !out->r_min || !out->n_acc ||
        !out->n_rej || !out->n_turn || !out->status || !out->complex_flag)
        return AIG_ERR_NULL;
    if (!aligned(y0, 8) || !aligned(workspace, 8) || !aligned(out->y_final, 8) || !aligned(out->t_final, 8) ||
        !aligned(out->lifetime, 8) || !aligned(out->angle, 8) || !aligned(out->r_min, 8) ||
        !aligned(out->n_acc, 4) || !aligned(out->n_rej, 4) || !aligned(out->n_turn, 4) ||
        !aligned(out->status, 4))
        return AIG_ERR_ALIGN;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const KParams K = make_kparams(p, t_max, rtol, atol);
    if (out->x_turn1) {
        if (!aligned(out->x_turn1, 8)) return AIG_ERR_ALIGN;
        // all-ones bytes = NaN: "no bounce, no position"; the kernels overwrite the rest once per trajectory
        if (cudaMemsetAsync(out->x_turn1, 0xFF, 3 * (size_t)N * sizeof(double), st) != cudaSuccess) return AIG_ERR_CUDA;
    }
    OutPtrs O{out->y_final, out->t_final, out->lifetime, out->angle, out->r_min,
              out->n_acc,   out->n_rej,   out->n_turn,   out->status, out->complex_flag, out->x_turn1};
    switch (trap_mode(p, t_max) + 4 * (general_potential(p) ? POT_GENERAL : POT_4_8)) {
        case TRAP_RF: return launch_integrate<TRAP_RF>(p, K, y0, N, O, workspace, st);
        case TRAP_RF_BIG: return launch_integrate<TRAP_RF_BIG>(p, K, y0, N, O, workspace, st);
        case TRAP_STATIC: return launch_integrate<TRAP_STATIC>(p, K, y0, N, O, workspace, st);
        case TRAP_NONE: return launch_integrate<TRAP_NONE>(p, K, y0, N, O, workspace, st);
        case 4 + TRAP_RF: return launch_integrate<4 + TRAP_RF>(p, K, y0, N, O, workspace, st);
        case 4 + TRAP_RF_BIG: return launch_integrate<4 + TRAP_RF_BIG>(p, K, y0, N, O, workspace, st);
        case 4 + TRAP_STATIC: return launch_integrate<4 + TRAP_STATIC>(p, K, y0, N, O, workspace, st);
        default: return launch_integrate<4 + TRAP_NONE>(p, K, y0, N, O, workspace, st);
    }
}

int aig_step_once(const aig_params* p, const double* y, const double* t, const double* h, int64_t N,
                  double rtol, double atol, double* ynew, double* err, void* cuda_stream)
{
    if (!p) return AIG_ERR_NULL;
    int rc = check_params(p, p->t0 + 1.0, rtol, atol);
    if (rc) return rc;
    if (N < 0 || N > (1LL << 40)) return AIG_ERR_SIZE;
    if (N == 0) return AIG_OK;
    if (!y || !t || !h || !ynew || !err) return AIG_ERR_NULL;
    if (!aligned(y, 8) || !aligned(t, 8) || !aligned(h, 8) || !aligned(ynew, 8) || !aligned(err, 8))
        return AIG_ERR_ALIGN;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    KParams K = make_kparams(p, p->t0 + 1.0, rtol, atol);
    K.t_max = INFINITY;
    const unsigned blocks = (unsigned)((N + kBlock - 1) / kBlock);
    switch (trap_mode(p, p->t0 + 1.0) + 4 * (general_potential(p) ? POT_GENERAL : POT_4_8)) {
        case TRAP_RF_BIG:
        case TRAP_RF: step_once_kernel<TRAP_RF><<<blocks, kBlock, 0, st>>>(K, y, t, h, N, ynew, err); break;
        case TRAP_STATIC: step_once_kernel<TRAP_STATIC><<<blocks, kBlock, 0, st>>>(K, y, t, h, N, ynew, err); break;
        case TRAP_NONE: step_once_kernel<TRAP_NONE><<<blocks, kBlock, 0, st>>>(K, y, t, h, N, ynew, err); break;
        case 4 + TRAP_RF_BIG:
        case 4 + TRAP_RF: step_once_kernel<4 + TRAP_RF><<<blocks, kBlock, 0, st>>>(K, y, t, h, N, ynew, err); break;
        case 4 + TRAP_STATIC: step_once_kernel<4 + TRAP_STATIC><<<blocks, kBlock, 0, st>>>(K, y, t, h, N, ynew, err); break;
        default: step_once_kernel<4 + TRAP_NONE><<<blocks, kBlock, 0, st>>>(K, y, t, h, N, ynew, err); break;
    }
    g_kernel_launches++;
    return cudaGetLastError() == cudaSuccess ? AIG_OK : AIG_ERR_CUDA;
}

int aig_histogram(const aig_out* obs, int64_t N, const aig_hist_spec* spec, const aig_hist* out,
                  void* cuda_stream)
{
    if (!obs || !spec || !out) return AIG_ERR_NULL;
    if (N < 0 || N > (1LL << 40)) return AIG_ERR_SIZE;
    if (spec->n_angle_bins < 1 || spec->n_life_bins < 1 || spec->n_turn_bins < 1) return AIG_ERR_SIZE;
    if (spec->n_angle_bins > 2048 || spec->n_life_bins > 2048 || spec->n_turn_bins > 2048) return AIG_ERR_SIZE;
    if (!spec->angle_edges || !spec->life_edges) return AIG_ERR_NULL;
    if (!out->angle || !out->lifetime || !out->n_turn || !out->status || !out->totals) return AIG_ERR_NULL;
    if (N == 0) return AIG_OK;
    if (!obs->angle || !obs->lifetime || !obs->n_acc || !obs->n_rej || !obs->n_turn || !obs->status ||
        !obs->complex_flag)
        return AIG_ERR_NULL;
    if (!aligned(spec->angle_edges, 8) || !aligned(spec->life_edges, 8) || !aligned(out->angle, 8) ||
        !aligned(out->lifetime, 8) || !aligned(out->n_turn, 8) || !aligned(out->status, 8) ||
        !aligned(out->totals, 8))
        return AIG_ERR_ALIGN;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    HistArgs a;
    a.angle = obs->angle;
    a.lifetime = obs->lifetime;
    a.n_acc = obs->n_acc;
    a.n_rej = obs->n_rej;
    a.n_turn = obs->n_turn;
    a.status = obs->status;
    a.complex_flag = obs->complex_flag;
    a.angle_edges = spec->angle_edges;
    a.life_edges = spec->life_edges;
    a.na = spec->n_angle_bins;
    a.nl = spec->n_life_bins;
    a.nt = spec->n_turn_bins;
    a.h_angle = reinterpret_cast<unsigned long long*>(out->angle);
    a.h_life = reinterpret_cast<unsigned long long*>(out->lifetime);
    a.h_turn = reinterpret_cast<unsigned long long*>(out->n_turn);
    a.h_status = reinterpret_cast<unsigned long long*>(out->status);
    a.h_totals = reinterpret_cast<unsigned long long*>(out->totals);
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return AIG_ERR_CUDA;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return AIG_ERR_CUDA;
    const size_t smem = sizeof(double) * (a.na + 1 + a.nl + 1) +
                        sizeof(unsigned) * ((a.na + 2) + (a.nl + 2) + a.nt + 4);
    long long blocks = (N + 255) / 256;
    const long long cap = (long long)sms * 8;
    if (blocks > cap) blocks = cap;
    histogram_kernel<<<(unsigned)blocks, 256, smem, st>>>(a, N);
    g_kernel_launches++;
    return cudaGetLastError() == cudaSuccess ? AIG_OK : AIG_ERR_CUDA;
}

int aig_trace(const aig_params* p, const double* y0, double t_max, double rtol, double atol, int64_t cap,
              double* t_out, double* y_out, int64_t* n_out, void* cuda_stream)
{
    int rc = check_params(p, t_max, rtol, atol);
    if (rc) return rc;
    if (cap < 0 || cap > (1LL << 40)) return AIG_ERR_SIZE;
    if (!y0 || !n_out || (cap > 0 && (!t_out || !y_out))) return AIG_ERR_NULL;
    if (!aligned(y0, 8) || !aligned(n_out, 8) || !aligned(t_out, 8) || !aligned(y_out, 8)) return AIG_ERR_ALIGN;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const KParams K = make_kparams(p, t_max, rtol, atol);
    long long* n = reinterpret_cast<long long*>(n_out);
    switch (trap_mode(p, t_max) + 4 * (general_potential(p) ? POT_GENERAL : POT_4_8)) {
        case TRAP_RF: trace_kernel<TRAP_RF><<<1, 32, 0, st>>>(K, y0, cap, t_out, y_out, n); break;
        case TRAP_RF_BIG: trace_kernel<TRAP_RF_BIG><<<1, 32, 0, st>>>(K, y0, cap, t_out, y_out, n); break;
        case TRAP_STATIC: trace_kernel<TRAP_STATIC><<<1, 32, 0, st>>>(K, y0, cap, t_out, y_out, n); break;
        case TRAP_NONE: trace_kernel<TRAP_NONE><<<1, 32, 0, st>>>(K, y0, cap, t_out, y_out, n); break;
        case 4 + TRAP_RF: trace_kernel<4 + TRAP_RF><<<1, 32, 0, st>>>(K, y0, cap, t_out, y_out, n); break;
        case 4 + TRAP_RF_BIG: trace_kernel<4 + TRAP_RF_BIG><<<1, 32, 0, st>>>(K, y0, cap, t_out, y_out, n); break;
        case 4 + TRAP_STATIC: trace_kernel<4 + TRAP_STATIC><<<1, 32, 0, st>>>(K, y0, cap, t_out, y_out, n); break;
        default: trace_kernel<4 + TRAP_NONE><<<1, 32, 0, st>>>(K, y0, cap, t_out, y_out, n); break;
    }
    g_kernel_launches++;
    return cudaGetLastError() == cudaSuccess ? AIG_OK : AIG_ERR_CUDA;
}

int aig_observables(const aig_params* p, const double* y0, const aig_out* out, int64_t N,
                    const aig_obs_extra* extra, void* cuda_stream)
{
    if (!p || !extra) return AIG_ERR_NULL;
    if (!(p->m_ion > 0.0) || !(p->m_atom > 0.0) || !std::isfinite(p->m_ion) || !std::isfinite(p->m_atom))
        return AIG_ERR_PARAM;
    if (N < 0 || N > (1LL << 40)) return AIG_ERR_SIZE;
    if (N == 0) return AIG_OK;
    if (!y0 || !out || !out->y_final || !extra->dist || !extra->KE || !extra->transfer) return AIG_ERR_NULL;
    if (extra->position && !out->x_turn1) return AIG_ERR_NULL;
    if (!aligned(y0, 8) || !aligned(out->y_final, 8) || !aligned(extra->dist, 8) || !aligned(extra->KE, 8) ||
        !aligned(extra->transfer, 8) || !aligned(extra->position, 8) || !aligned(out->x_turn1, 8))
        return AIG_ERR_ALIGN;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return AIG_ERR_CUDA;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return AIG_ERR_CUDA;
    const long long blocks = std::min<long long>((N + 255) / 256, (long long)sms * 8);
    observables_kernel<<<(unsigned)blocks, 256, 0, static_cast<cudaStream_t>(cuda_stream)>>>(
        y0, out->y_final, N, p->m_ion, p->m_atom, extra->dist, extra->KE, extra->transfer, out->x_turn1, extra->position);
    g_kernel_launches++;
    return cudaGetLastError() == cudaSuccess ? AIG_OK : AIG_ERR_CUDA;
}

constexpr int kOutlierBlocksMax = 1024;

size_t aig_outliers_workspace_bytes(void)
{
    return 256 + (size_t)kOutlierBlocksMax * kOutlierObs * 2 * sizeof(Extreme);
}

int aig_outliers(const aig_out* out, const aig_obs_extra* extra, int64_t N, int64_t* result, void* workspace,
                 void* cuda_stream)
{
    if (!result || !workspace) return AIG_ERR_NULL;
    if (N < 0 || N > (1LL << 40)) return AIG_ERR_SIZE;
    if (!aligned(result, 8) || !aligned(workspace, 16)) return AIG_ERR_ALIGN;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    if (N > 0) {
        if (!out || !extra) return AIG_ERR_NULL;
        if (!out->angle || !out->lifetime || !out->n_turn || !out->n_acc || !extra->dist || !extra->KE || !extra->transfer)
            return AIG_ERR_NULL;
    }
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return AIG_ERR_CUDA;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return AIG_ERR_CUDA;
    if (cudaMemsetAsync(workspace, 0, 256, st) != cudaSuccess) return AIG_ERR_CUDA;
    OutlierArgs a;
    a.angle = N ? out->angle : nullptr;
    a.lifetime = N ? out->lifetime : nullptr;
    a.n_turn = N ? out->n_turn : nullptr;
    a.n_acc = N ? out->n_acc : nullptr;
    a.transfer = N ? extra->transfer : nullptr;
    a.dist = N ? extra->dist : nullptr;
    a.ke = N ? extra->KE : nullptr;
    a.position = N ? extra->position : nullptr;
    a.ticket = static_cast<unsigned int*>(workspace);
    a.partial = reinterpret_cast<Extreme*>(static_cast<unsigned char*>(workspace) + 256);
    a.result = reinterpret_cast<long long*>(result);
    int occ = 0;  // one wave of resident blocks: the last block to finish folds the partials
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, outliers_kernel, 256, 0) != cudaSuccess || occ < 1) return AIG_ERR_CUDA;
    long long blocks = std::min<long long>(std::max<long long>(1, (N + 255) / 256), std::min<long long>((long long)sms * occ, kOutlierBlocksMax));
    outliers_kernel<<<(unsigned)blocks, 256, 0, st>>>(a, N);
    g_kernel_launches++;
    return cudaGetLastError() == cudaSuccess ? AIG_OK : AIG_ERR_CUDA;
}

int aig_run_host(const aig_params* p, const double* y0_host, int64_t N, double t_max, double rtol,
                 double atol, const aig_out* out_host, const aig_hist_spec* hs, const aig_hist* ho)
{
    int rc = check_params(p, t_max, rtol, atol);
    if (rc) return rc;
    if (N < 0 || N > (1LL << 40)) return AIG_ERR_SIZE;
    if (!y0_host || !out_host) return AIG_ERR_NULL;
    if ((hs == nullptr) != (ho == nullptr)) return AIG_ERR_NULL;
    if (N == 0) return AIG_OK;
    const size_t n = (size_t)N;
    // one device slab: y0 | y_final | 4 double arrays | 4 int arrays | flag | workspace | hist
    const size_t b_y = 12 * n * sizeof(double), b_d = n * sizeof(double), b_i = n * sizeof(int32_t);
    size_t hist_words = 0, edge_words = 0;
    if (hs) {
        if (hs->n_angle_bins < 1 || hs->n_life_bins < 1 || hs->n_turn_bins < 1) return AIG_ERR_SIZE;
        if (!hs->angle_edges || !hs->life_edges) return AIG_ERR_NULL;
        hist_words = (size_t)(hs->n_angle_bins + 2) + (hs->n_life_bins + 2) + hs->n_turn_bins + 4 + 4;
        edge_words = (size_t)(hs->n_angle_bins + 1) + (hs->n_life_bins + 1);
    }
    const size_t flag_bytes = (n + 255) / 256 * 256;
    const size_t ws_bytes = round_up(aig_workspace_bytes(N), 256);
    const size_t b_x = out_host->x_turn1 ? 3 * b_d : 0;
    const size_t total = 2 * b_y + 4 * b_d + b_x + 4 * b_i + flag_bytes + ws_bytes + 8 * (hist_words + edge_words) + 8192;
    unsigned char* slab = nullptr;
    cudaStream_t st = nullptr;
    if (cudaMalloc(&slab, total) != cudaSuccess) return AIG_ERR_CUDA;
    auto fail = [&](int code) {
        cudaDeviceSynchronize();
        cudaFree(slab);
        (void)cudaGetLastError();
        return code;
    };
    unsigned char* cur = slab;
    auto take = [&](size_t bytes) {
        unsigned char* r = cur;
        cur += (bytes + 255) / 256 * 256;
        return r;
    };
    double* d_y0 = reinterpret_cast<double*>(take(b_y));
    aig_out d;
    d.y_final = reinterpret_cast<double*>(take(b_y));
    d.t_final = reinterpret_cast<double*>(take(b_d));
    d.lifetime = reinterpret_cast<double*>(take(b_d));
    d.angle = reinterpret_cast<double*>(take(b_d));
    d.r_min = reinterpret_cast<double*>(take(b_d));
    d.n_acc = reinterpret_cast<int32_t*>(take(b_i));
    d.n_rej = reinterpret_cast<int32_t*>(take(b_i));
    d.n_turn = reinterpret_cast<int32_t*>(take(b_i));
    d.status = reinterpret_cast<int32_t*>(take(b_i));
    d.complex_flag = take(flag_bytes);
    d.x_turn1 = b_x ? reinterpret_cast<double*>(take(b_x)) : nullptr;
    void* ws = take(ws_bytes);
    if (cudaMemcpyAsync(d_y0, y0_host, b_y, cudaMemcpyHostToDevice, st) != cudaSuccess) return fail(AIG_ERR_CUDA);
    rc = aig_integrate(p, d_y0, N, t_max, rtol, atol, &d, ws, st);
    if (rc) return fail(rc);
    uint64_t* d_hist = nullptr;
    if (hs) {
        d_hist = reinterpret_cast<uint64_t*>(take(8 * hist_words));
        double* d_edges = reinterpret_cast<double*>(take(8 * edge_words));
        if (cudaMemsetAsync(d_hist, 0, 8 * hist_words, st) != cudaSuccess) return fail(AIG_ERR_CUDA);
        if (cudaMemcpyAsync(d_edges, hs->angle_edges, 8 * (hs->n_angle_bins + 1), cudaMemcpyHostToDevice, st) !=
                cudaSuccess ||
            cudaMemcpyAsync(d_edges + hs->n_angle_bins + 1, hs->life_edges, 8 * (hs->n_life_bins + 1),
                            cudaMemcpyHostToDevice, st) != cudaSuccess)
            return fail(AIG_ERR_CUDA);
        aig_hist_spec ds = *hs;
        ds.angle_edges = d_edges;
        ds.life_edges = d_edges + hs->n_angle_bins + 1;
        aig_hist dh;
        dh.angle = d_hist;
        dh.lifetime = dh.angle + hs->n_angle_bins + 2;
        dh.n_turn = dh.lifetime + hs->n_life_bins + 2;
        dh.status = dh.n_turn + hs->n_turn_bins;
        dh.totals = dh.status + 4;
        rc = aig_histogram(&d, N, &ds, &dh, st);
        if (rc) return fail(rc);
        const cudaMemcpyKind D2H = cudaMemcpyDeviceToHost;
        bool ok = true;
        if (ho->angle) ok = ok && cudaMemcpyAsync(ho->angle, dh.angle, 8 * (hs->n_angle_bins + 2), D2H, st) == cudaSuccess;
        if (ho->lifetime) ok = ok && cudaMemcpyAsync(ho->lifetime, dh.lifetime, 8 * (hs->n_life_bins + 2), D2H, st) == cudaSuccess;
        if (ho->n_turn) ok = ok && cudaMemcpyAsync(ho->n_turn, dh.n_turn, 8 * hs->n_turn_bins, D2H, st) == cudaSuccess;
        if (ho->status) ok = ok && cudaMemcpyAsync(ho->status, dh.status, 8 * 4, D2H, st) == cudaSuccess;
        if (ho->totals) ok = ok && cudaMemcpyAsync(ho->totals, dh.totals, 8 * 4, D2H, st) == cudaSuccess;
        if (!ok) return fail(AIG_ERR_CUDA);
    }
    {
        const cudaMemcpyKind D2H = cudaMemcpyDeviceToHost;
        bool ok = true;
        const aig_out* o = out_host;
        if (o->y_final) ok = ok && cudaMemcpyAsync(o->y_final, d.y_final, b_y, D2H, st) == cudaSuccess;
        if (o->t_final) ok = ok && cudaMemcpyAsync(o->t_final, d.t_final, b_d, D2H, st) == cudaSuccess;
        if (o->lifetime) ok = ok && cudaMemcpyAsync(o->lifetime, d.lifetime, b_d, D2H, st) == cudaSuccess;
        if (o->angle) ok = ok && cudaMemcpyAsync(o->angle, d.angle, b_d, D2H, st) == cudaSuccess;
        if (o->r_min) ok = ok && cudaMemcpyAsync(o->r_min, d.r_min, b_d, D2H, st) == cudaSuccess;
        if (o->n_acc) ok = ok && cudaMemcpyAsync(o->n_acc, d.n_acc, b_i, D2H, st) == cudaSuccess;
        if (o->n_rej) ok = ok && cudaMemcpyAsync(o->n_rej, d.n_rej, b_i, D2H, st) == cudaSuccess;
        if (o->n_turn) ok = ok && cudaMemcpyAsync(o->n_turn, d.n_turn, b_i, D2H, st) == cudaSuccess;
        if (o->status) ok = ok && cudaMemcpyAsync(o->status, d.status, b_i, D2H, st) == cudaSuccess;
        if (o->complex_flag) ok = ok && cudaMemcpyAsync(o->complex_flag, d.complex_flag, n, D2H, st) == cudaSuccess;
        if (o->x_turn1) ok = ok && cudaMemcpyAsync(o->x_turn1, d.x_turn1, b_x, D2H, st) == cudaSuccess;
        if (!ok) return fail(AIG_ERR_CUDA);
    }
    if (cudaStreamSynchronize(st) != cudaSuccess) return fail(AIG_ERR_CUDA);
    cudaFree(slab);
    return AIG_OK;
}

int aig_fp64_peak_probe(int iters, int ilp, double* flops_per_s, double* elapsed_ms)
{
    if (!flops_per_s) return AIG_ERR_NULL;
    if (iters < 1 || ilp < 1 || ilp > 16) return AIG_ERR_SIZE;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return AIG_ERR_CUDA;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return AIG_ERR_CUDA;
    double* d_out = nullptr;
    if (cudaMalloc(&d_out, 8) != cudaSuccess) return AIG_ERR_CUDA;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const int blocks = sms * 8, threads = 256;
    int used = ilp >= 16 ? 16 : (ilp >= 8 ? 8 : (ilp >= 4 ? 4 : (ilp >= 2 ? 2 : 1)));
    auto launch = [&](int it) {
        switch (used) {
            case 16: dfma_probe_kernel<16><<<blocks, threads>>>(d_out, it, 0.999999, 1e-6); break;
            case 8: dfma_probe_kernel<8><<<blocks, threads>>>(d_out, it, 0.999999, 1e-6); break;
            case 4: dfma_probe_kernel<4><<<blocks, threads>>>(d_out, it, 0.999999, 1e-6); break;
            case 2: dfma_probe_kernel<2><<<blocks, threads>>>(d_out, it, 0.999999, 1e-6); break;
            default: dfma_probe_kernel<1><<<blocks, threads>>>(d_out, it, 0.999999, 1e-6); break;
        }
    };
    launch(iters / 8 + 1);  // warm-up
    cudaEventRecord(e0);
    launch(iters);
    cudaEventRecord(e1);
    int rc = AIG_OK;
    if (cudaEventSynchronize(e1) != cudaSuccess || cudaGetLastError() != cudaSuccess) rc = AIG_ERR_CUDA;
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(d_out);
    if (rc) return rc;
    const double flops = 2.0 * 8.0 * used * (double)iters * (double)blocks * threads;
    *flops_per_s = flops / (ms * 1e-3);
    if (elapsed_ms) *elapsed_ms = ms;
    return AIG_OK;
}

int aig_kernel_info(int* sm_count, int* blocks_per_sm, int* threads_per_block, int* regs_per_thread,
                    int* local_bytes_per_thread)
{
    cudaFuncAttributes fa;
    if (cudaFuncGetAttributes(&fa, integrate_kernel<TRAP_RF, kBlock, kBlocksPerSM>) != cudaSuccess) return AIG_ERR_CUDA;
    int bps = 0, sms = 0;
    const int rc = bulk_capacity<TRAP_RF>(&bps, &sms);
    if (rc) return rc;
    if (sm_count) *sm_count = sms;
    if (blocks_per_sm) *blocks_per_sm = bps;
    if (threads_per_block) *threads_per_block = kBlock;
    if (regs_per_thread) *regs_per_thread = fa.numRegs;
    if (local_bytes_per_thread) *local_bytes_per_thread = (int)fa.localSizeBytes;
    return AIG_OK;
}

}  // extern "C"
