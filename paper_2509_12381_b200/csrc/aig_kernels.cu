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
#define AIG_MIN_BLOCKS 3
#endif
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
// Cold state of the per-thread integrator: shared memory, one 8-byte slot per thread and row, every row
// at a compile-time offset from ONE per-thread address (a separate array each would cost an address
// register each: the kernel runs at the 168 registers that allow three blocks per SM).
//   rows: 0 r_min^2, 1 t_first, 2 t_last, 3 (n_rej, n_turn), 4-6 initial atom velocity, 7 trajectory index,
//         8 (accepted steps at which the trajectory is offered next, iterations an idle lane of the warp has waited),
//         9 (iterations since the queue was seen empty, stop status of a finished trajectory not stored yet),
//         10 the radial observable s(t) between two steps (Core::sprev: read and written once per step),
//         11 (accepted steps, flags) between two steps (Core::n_acc, Core::flags: likewise)
constexpr int kColdRows = 12;
template <int BLOCK>
struct ColdShared {
    static constexpr bool kInRegisters = false;
    double* b;  // row 0 of this thread
    __device__ __forceinline__ double& rmin2() { return b[0 * BLOCK]; }
    __device__ __forceinline__ double& t_first() { return b[1 * BLOCK]; }
    __device__ __forceinline__ double& t_last() { return b[2 * BLOCK]; }
    __device__ __forceinline__ int& n_rej() { return reinterpret_cast<int*>(b + 3 * BLOCK)[0]; }
    __device__ __forceinline__ int& n_turn() { return reinterpret_cast<int*>(b + 3 * BLOCK)[1]; }
    __device__ __forceinline__ double& v0(int k) { return b[(4 + k) * BLOCK]; }
    __device__ __forceinline__ long long& idx() { return *reinterpret_cast<long long*>(b + 7 * BLOCK); }
    __device__ __forceinline__ int& stop_at() { return reinterpret_cast<int*>(b + 8 * BLOCK)[0]; }
    __device__ __forceinline__ int& waited() { return reinterpret_cast<int*>(b + 8 * BLOCK)[1]; }
    __device__ __forceinline__ int& since_dry() { return reinterpret_cast<int*>(b + 9 * BLOCK)[0]; }
    __device__ __forceinline__ int& pending() { return reinterpret_cast<int*>(b + 9 * BLOCK)[1]; }
    __device__ __forceinline__ double& sprev() { return b[10 * BLOCK]; }
    __device__ __forceinline__ volatile int& n_acc() { return reinterpret_cast<volatile int*>(b + 11 * BLOCK)[0]; }
    __device__ __forceinline__ volatile int& flags() { return reinterpret_cast<volatile int*>(b + 11 * BLOCK)[1]; }
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
//           18 t, 19 h, 20 s(t), 21 r_min^2, 22 t_first, 23 t_last;  i rows: n_acc, flags, n_rej, n_turn,
//           time of the hand-over (two rows; diagnostics)
struct Ckpt {
    double* d;
    int* i;
    long long* idx;
    long long cap;
};
constexpr int kCkptDoubles = 24, kCkptInts = 6;  // i rows 4, 5: %globaltimer of the hand-over (diagnostics)
constexpr size_t kCkptBytesPerSlot = kCkptDoubles * 8 + kCkptInts * 4 + 8;

__device__ __forceinline__ unsigned long long ld_volatile(const unsigned long long* p)
{
    return *(const volatile unsigned long long*)p;
}

// A slot is PUBLISHED by its idx entry: the entries are -1 when the call starts (memset), the writer
// stores every field, fences, and stores the trajectory index last; a reader that has claimed the slot
// number spins on idx >= 0, fences, and reads the fields past L1 (ckpt_wait / __ldcg).
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
    const unsigned long long now = global_ns();
    q[4 * cap] = (int)(unsigned)(now & 0xffffffffULL);
    q[5 * cap] = (int)(unsigned)(now >> 32);
    __threadfence();
    *(volatile long long*)(K.idx + slot) = idx;
}

// trajectory index of a claimed slot, once its writer has published it.  The writer took the slot number
// while running and publishes within microseconds.  %globaltimer is wall time and keeps running while the
// context is time-sliced, preempted or replayed by a profiler, so the limit that turns a broken invariant
// into a loud failure (a trap poisons the context: the whole call is lost) rather than a hang is generous:
// thirty seconds without the writer is not scheduling noise.
constexpr unsigned long long kCkptWaitLimitNs = 30000000000ULL;
__device__ __forceinline__ long long ckpt_wait(const Ckpt& K, long long slot)
{
    long long idx = *(const volatile long long*)(K.idx + slot);
    if (idx < 0) {
        const unsigned long long t0 = global_ns();
        while ((idx = *(const volatile long long*)(K.idx + slot)) < 0) {
            __nanosleep(100);
            if (global_ns() - t0 > kCkptWaitLimitNs) __trap();
        }
    }
    __threadfence();
    return idx;
}

// Scheduling arguments of one launch of the per-thread integrator.  Work items are the entries
// [*begin, *end) of `order` (trajectory indices; order == nullptr: the indices themselves).  A lane
// whose trajectory has not ended is suspended -- its state written to slot atomicAdd(*n_out, 1) of
// `out` and published there, for the six-lane integrator that runs BESIDE this kernel and takes slots
// as they appear (*taken = slots it has claimed so far) --
//   (a) when it has taken `budget` accepted steps, is `mean_factor` times longer than the mean of the
//       trajectories this launch has finished (a workload in which every trajectory is long is this
//       kernel's job: nothing is handed over before 32 have finished), has reached the BAR, and the
//       six-lane pass has room: fewer than its capacity + `depth` trajectories handed over and not yet
//       finished (it has less than half the throughput per FP64 operation: it is for the few, and a
//       suspended trajectory that waits makes no progress).  The bar is a feedback loop: a trajectory
//       at or above it that is refused for lack of room nudges it up (by 1/64, at most once per 20 us)
//       and asks again 64 steps later; the six-lane pass nudges it down while a quarter of its groups
//       are idle.  It settles where the trajectories that cross it arrive as fast as the six-lane pass
//       finishes others: the fast lane then holds the LONGEST-running trajectories, which is what
//       bounds the end of the call.  A trajectory below the bar is asked again at the bar, or one
//       budget later; or
//   (b) when, `tail_iters` iterations after its warp has seen the queue empty, the warp has
//       `drain_lanes` or fewer trajectories left.
// When the slots are exhausted it simply keeps stepping.  Suspension never changes a trajectory's
// arithmetic, only where it continues.
struct Sched {
    unsigned long long* queue;
    const long long* order;
    const unsigned long long *begin, *end;
    unsigned long long* n_out;
    const unsigned long long* finished;  // trajectories the six-lane passes have finished
    unsigned long long* bar;             // accepted steps a trajectory must have to be offered (see below)
    long long capacity;                  // trajectories the streaming six-lane pass can step at once
    unsigned long long* started;     // set to 1 by the first block to run
    unsigned long long* done_warps;  // warps that have exited (the six-lane pass beside this kernel ends when all have)
    Ckpt out;
    int depth;
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
    __shared__ double s_cold[kColdRows][BLOCK];
    ColdShared<BLOCK> C{&s_cold[0][threadIdx.x]};
    const unsigned FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    // the queue's range: block-wide constants of the refill code only, kept out of the registers
    __shared__ long long s_range[2];
    if (threadIdx.x == 0) {
        s_range[0] = (long long)*S.begin;
        s_range[1] = (long long)*S.end - s_range[0];
    }
    __syncthreads();
    if (blockIdx.x == 0 && threadIdx.x == 0) *(volatile unsigned long long*)S.started = 1ULL;
    Traj T;
    C.idx() = -1;
    C.waited() = 0;     // warp-uniform: iterations since a lane of this warp went idle
    C.since_dry() = 0;  // warp-uniform: iterations since the queue was seen empty
    C.pending() = -1;   // stop status of a finished trajectory whose results are not stored yet
    bool live = false;
    bool dry = false;     // warp-uniform: the queue has been seen empty
    bool may_suspend = true;
    stage_begin(S.timeline);

    for (;;) {
        // ---- service: lanes without a trajectory store what they finished and take the next items
        //      of the queue.  The whole warp walks through this code (atan2 / sqrt of the end, global
        //      loads and the twelve divisions of the start) whenever one lane needs it, so idle lanes
        //      are served in batches: when refill_batch of them wait, or one has C.waited() refill_wait
        //      iterations, or the queue is empty.
        const unsigned need = __ballot_sync(FULL, !live);
        if (need && (__popc(need) >= S.refill_batch || C.waited() >= S.refill_wait || dry)) {
            C.waited() = 0;
            {   // accepted steps and count of what this warp has finished since its last service
                const unsigned fm = __ballot_sync(FULL, C.pending() >= 0);
                if (fm) {
                    const unsigned steps = __reduce_add_sync(FULL, C.pending() >= 0 ? (unsigned)T.c.n_acc : 0u);
                    if (lane == 0) {
                        atomicAdd(S.stats + 0, (unsigned long long)steps);
                        atomicAdd(S.stats + 1, (unsigned long long)__popc(fm));
                    }
                }
            }
            if (C.pending() >= 0) {
                const double v0[3] = {C.v0(0), C.v0(1), C.v0(2)};
                store_traj(v0, N, C.idx(), T, C, C.pending(), O);
                C.pending() = -1;
            }
            if (!dry) {
                const long long first = s_range[0], total = s_range[1];
                const int cnt = __popc(need);
                const int leader = __ffs(need) - 1;
                unsigned long long base = 0;
                if (lane == leader) base = atomicAdd(S.queue, (unsigned long long)cnt);
                base = __shfl_sync(FULL, base, leader);
                if (!live) {
                    const long long cand = (long long)base + __popc(need & ((1u << lane) - 1u));
                    if (cand < total) {
                        const long long idx = S.order ? S.order[first + cand] : first + cand;
                        C.idx() = idx;
                        load_traj<TRAP>(P, y0, N, idx, T, C);
                        C.sprev() = T.c.sprev;
                        C.n_acc() = T.c.n_acc;
                        C.flags() = (int)T.c.flags;
#pragma unroll
                        for (int k = 0; k < 3; ++k) C.v0(k) = T.V[3 + k];
                        C.stop_at() = S.budget;
                        may_suspend = true;
                        live = true;
                    }
                }
                if ((long long)base + cnt >= total) dry = true;
            }
            if (!__any_sync(FULL, live)) break;
        } else if (need) {
            ++C.waited();
        }
        // warp-uniform: the queue is empty, the grace period is over and few lanes are still alive: at
        // fewer than ~11 lanes the six-lane kernel does more steps per SM and second than this one
        const bool drain = dry && C.since_dry() > S.tail_iters && (32 - __popc(need)) <= S.drain_lanes;
        if (dry) ++C.since_dry();
        // ---- one attempted step for every live lane
        if (live) {
            // s(t), the step counter and the flags live in shared memory between two steps (volatile: re-read, not
            // kept): three registers less through the stages, which is what lets the kernel run at 168 without a spill
            Attempt R;
            T.c.flags = (unsigned)C.flags();
            dp45_attempt<TRAP>(P, T, R);
            bool first_turn;
            T.c.sprev = C.sprev();
            T.c.n_acc = C.n_acc();
            T.c.flags = (unsigned)C.flags();
            const int st = finish_attempt(P, T, C, R, first_turn);
            C.sprev() = T.c.sprev;
            C.n_acc() = T.c.n_acc;
            C.flags() = (int)T.c.flags;
            if (first_turn && O.x_turn1) {  // once per trajectory ("position")
#pragma unroll
                for (int k = 0; k < 3; ++k) O.x_turn1[k * N + C.idx()] = T.X[k];
            }
            if (st >= 0) {
                C.pending() = st;
                live = false;
            } else if (may_suspend && (T.c.n_acc >= C.stop_at() || drain)) {
                bool room = true;
                if (!drain) {
                    // budget hand-over: only while few published slots wait to be taken, and only for a
                    // trajectory that is long compared with what this launch has finished so far
                    const unsigned long long n_now = (unsigned long long)T.c.n_acc;
                    const unsigned long long bar = ld_volatile(S.bar);
                    int again = S.budget;  // steps until the next offer
                    room = n_now >= bar;
                    if (!room && bar - n_now < (unsigned long long)again) again = (int)(bar - n_now);
                    if (room && S.mean_factor > 0) {
                        const unsigned long long cnt = *(volatile unsigned long long*)(S.stats + 1);
                        const unsigned long long sum = *(volatile unsigned long long*)(S.stats + 0);
                        room = (cnt >= 32ULL) && (n_now * cnt >= (unsigned long long)S.mean_factor * sum);
                    }
                    if (room) {
                        const unsigned long long fin = ld_volatile(S.finished), out = ld_volatile(S.n_out);
                        room = out < fin + (unsigned long long)(S.capacity + S.depth);
                        if (!room) {
                            again = 64;
                            const unsigned long long now = global_ns(), last = ld_volatile(S.bar + 1);
                            if (now - last > 20000ULL && atomicCAS(S.bar + 1, last, now) == last) {
                                const unsigned long long b = bar > (unsigned long long)S.budget ? bar : (unsigned long long)S.budget;
                                *(volatile unsigned long long*)S.bar = b + (b >> 6) + 1ULL;
                            }
                        }
                    }
                    if (!room) C.stop_at() = T.c.n_acc + again;
                }
                if (room) {
                    const long long slot = (long long)atomicAdd(S.n_out, 1ULL);
                    if (slot < S.out.cap) {
                        ckpt_store(S.out, slot, C.idx(), T, C);
                        live = false;
                    } else {
                        may_suspend = false;  // no slot left: finish it here
                    }
                }
            }
        }
    }
    stage_end(S.timeline);
    __threadfence();  // this warp's slots are published before it counts as done
    if (lane == 0) atomicAdd(S.done_warps, 1ULL);
}

// ---- six lanes per trajectory: continues published checkpoint slots to their end.  Slots are taken
// in the order they were handed out, by whichever pass asks first (*taken is the shared queue head,
// advanced by compare-and-swap up to the number handed out so far).  A pass either runs BESIDE the
// per-thread integrator (streaming: it polls for new slots and ends when every warp of that kernel
// has exited and every slot is taken) or after it (the final pass: the same code, nothing to wait for).
// Waiting is one-sided -- the per-thread integrator never waits for this kernel -- and bounded: a
// streaming pass that does not see the per-thread integrator START within `patience_ns` (kernels
// serialised by a profiler, a busy device) leaves, and what it would have done is done by the final pass.
struct SplitSched {
    unsigned long long* timeline;
    unsigned long long* loaded;            // diagnostics: trajectories this pass has taken
    unsigned long long* taken;             // queue head: slots [0, *taken) are claimed
    const unsigned long long* n_out;       // slots handed out so far (may overshoot the capacity)
    const unsigned long long* started;     // != 0 once the per-thread integrator of this call runs
    const unsigned long long* done_warps;  // warps of it that have exited ...
    unsigned long long producer_warps;     // ... of this many
    unsigned long long patience_ns;
    int poll_iters;                        // a warp with idle groups looks for new slots every this many iterations
    unsigned long long* finished;          // trajectories finished by the six-lane passes
    unsigned long long* bar;               // the hand-over bar (Sched); lowered here while groups are idle
    unsigned long long bar_floor;          // ... down to this (the budget)
    long long capacity;                    // groups of the streaming pass (0: this pass does not touch the bar)
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
    const unsigned long long cap = (unsigned long long)S.in.cap;
    SplitState Y;
    Core K;
    ColdRegs C;
    C.rmin2_ = C.t_first_ = C.t_last_ = 0.0;
    C.n_rej_ = C.n_turn_ = 0;
    long long idx = -1;
    bool live = false;

    // refill: every idle group takes the next published slot (one compare-and-swap per warp)
    auto refill = [&]() {
        const unsigned need = __ballot_sync(FULL, leader && !live);
        if (need == 0u) return;
        const int cnt = __popc(need);
        unsigned long long base = 0;
        int got = 0;
        if (lane == 0) {
            for (;;) {
                const unsigned long long head = ld_volatile(S.taken);
                unsigned long long avail = ld_volatile(S.n_out);
                avail = avail < cap ? avail : cap;
                if (head >= avail) {
                    // nothing waits.  One warp of the streaming pass nudges the bar down (by 1/64, at most once per
                    // 20 us) while a quarter of the groups are idle (plain stores: a lost update only delays the next)
                    if (S.capacity > 0 && blockIdx.x == 0 && threadIdx.x == 0) {
                        const unsigned long long busy = head - ld_volatile(S.finished);
                        const unsigned long long bar = ld_volatile(S.bar);
                        const unsigned long long now = global_ns();
                        if (4 * busy < 3 * (unsigned long long)S.capacity && bar > S.bar_floor && now - ld_volatile(S.bar + 1) > 20000ULL) {
                            const unsigned long long lower = bar - (bar >> 6) - 1ULL;
                            *(volatile unsigned long long*)S.bar = lower > S.bar_floor ? lower : S.bar_floor;
                            *(volatile unsigned long long*)(S.bar + 1) = now;
                        }
                    }
                    break;
                }
                const unsigned long long want = (avail - head) < (unsigned long long)cnt ? (avail - head) : (unsigned long long)cnt;
                if (atomicCAS(S.taken, head, head + want) == head) {
                    base = head;
                    got = (int)want;
                    atomicAdd(S.loaded, want);
                    break;
                }
            }
        }
        got = __shfl_sync(FULL, got, 0);
        base = __shfl_sync(FULL, base, 0);
        if (got == 0) return;
        if (!R.ghost && ((need >> R.base) & 1u)) {
            const int rank = __popc(need & ((1u << R.base) - 1u));
            if (rank < got) {
                const long long slot = (long long)base + rank;
                idx = ckpt_wait(S.in, slot);
                const double* d = S.in.d + slot;
                Y.xi = __ldcg(d + (0 + R.k) * cap);
                Y.xa = __ldcg(d + (3 + R.k) * cap);
                Y.vi = __ldcg(d + (6 + R.k) * cap);
                Y.va = __ldcg(d + (9 + R.k) * cap);
                Y.a1i = __ldcg(d + (12 + R.k) * cap);
                Y.a1a = __ldcg(d + (15 + R.k) * cap);
                K.t = __ldcg(d + 18 * cap);
                K.h = __ldcg(d + 19 * cap);
                K.sprev = __ldcg(d + 20 * cap);
                C.rmin2_ = __ldcg(d + 21 * cap);
                C.t_first_ = __ldcg(d + 22 * cap);
                C.t_last_ = __ldcg(d + 23 * cap);
                const int* q = S.in.i + slot;
                K.n_acc = __ldcg(q + 0 * cap);
                K.flags = (unsigned)__ldcg(q + 1 * cap);
                C.n_rej_ = __ldcg(q + 2 * cap);
                C.n_turn_ = __ldcg(q + 3 * cap);
                live = true;
            }
        }
    };

    // state of a group without a trajectory: it takes part in every shuffle and, in the fast loop below, steps
    // freely (an ion alone in the trap, the atom out of reach); nothing of it is ever stored
    auto park = [&]() {
        Y.xi = 1.0 + R.k;
        Y.xa = 1.0e6 * (1.0 + R.k);
        Y.vi = Y.va = Y.a1i = Y.a1a = 0.0;
        K.t = P.t0;
        K.h = 1.0;
        K.sprev = 0.0;
        K.n_acc = 0;
        K.flags = 0u;
    };
    park();

    stage_begin(S.timeline);
    const unsigned long long t_begin = global_ns();
    for (;;) {
        if (!__any_sync(FULL, live)) {
            // ---- nothing to step: take new slots, or find out that there will be none
            refill();
            if (!__any_sync(FULL, live)) {
                int leave = 0;
                if (lane == 0) {
                    const unsigned long long now = global_ns();
                    if (ld_volatile(S.done_warps) >= S.producer_warps) {
                        __threadfence();
                        unsigned long long avail = ld_volatile(S.n_out);
                        avail = avail < cap ? avail : cap;
                        leave = ld_volatile(S.taken) >= avail;
                    } else if (ld_volatile(S.started) == 0ULL) {
                        leave = (now - t_begin > S.patience_ns);
                    } else {
                        leave = (now - t_begin > 120000000000ULL);  // two minutes: never in practice
                    }
                }
                if (__shfl_sync(FULL, leave, 0)) break;
                __nanosleep(500);
                continue;
            }
        }
        // ---- fast loop: one attempted step of every group per iteration (all lanes together: full-mask
        //      shuffles inside).  As long as every trajectory of the warp takes the common case (accepted,
        //      nothing else happens: fast_step_ok) the loop body is ONE basic block -- commit, next attempt,
        //      vote -- so that the step-size chain of one step continues into the next and the instruction
        //      scheduler orders the bookkeeping behind it.  Groups without a trajectory never veto.  A warp
        //      with idle groups leaves the loop every poll_iters steps to look for new slots.
        const bool has_idle = __any_sync(FULL, leader && !live);
        int since_poll = 0;
        SplitAttempt A, B;
        split_attempt<TRAP>(P, R, K, Y, A);
        // two steps per iteration (A, B alternate): no register moves between the steps
        for (;;) {
            const bool okA = (!live | fast_step_ok(P, K, A.q_own, A.t_new, A.r2, A.s)) &
                             !(has_idle & (++since_poll > S.poll_iters));
            if (!__all_sync(FULL, okA)) break;
            fast_step_commit(P, K, C, A.err, A.t_new, A.r2, A.s);
            Y = A.Y;
            split_attempt<TRAP>(P, R, K, Y, B);
            const bool okB = !live | fast_step_ok(P, K, B.q_own, B.t_new, B.r2, B.s);
            if (!__all_sync(FULL, okB)) {
                A = B;
                break;
            }
            fast_step_commit(P, K, C, B.err, B.t_new, B.r2, B.s);
            Y = B.Y;
            split_attempt<TRAP>(P, R, K, Y, A);
        }
        // ---- the general case, one step: rejections, turning points, stops (finish_core)
        int st;
        {
            const StepTimes ST = step_times(P, K);
            const double err = A.finite ? A.err : __longlong_as_double(0x7ff8000000000000LL);
            bool accepted, first_turn;
            st = finish_core(P, K, C, err, ST, A.r2, A.s, live, accepted, first_turn);
            // once per trajectory ("position"): lane (k, 0) holds component k of the ion
            if (first_turn && R.e == 0 && O.x_turn1) O.x_turn1[R.k * N + idx] = A.Y.xi;
            Y.xi = accepted ? A.Y.xi : Y.xi;
            Y.vi = accepted ? A.Y.vi : Y.vi;
            Y.a1i = accepted ? A.Y.a1i : Y.a1i;
            Y.xa = accepted ? A.Y.xa : Y.xa;
            Y.va = accepted ? A.Y.va : Y.va;
            Y.a1a = accepted ? A.Y.a1a : Y.a1a;
        }
        const unsigned fin = __ballot_sync(FULL, st >= 0);
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
                atomicAdd(S.finished, 1ULL);
            }
            live = false;
            park();
        }
        if (fin != 0u || has_idle) refill();
    }
    stage_end(S.timeline);
}

// ---- work-queue order: the trajectories that can become long first ------------------------------
// (1) A trajectory can only form a complex (orders of magnitude more steps) if it gets over the
//     centrifugal barrier of the -C4/r^4 tail, i.e. if the atom passes the ion within the Langevin
//     radius b_c = (4 C4/E)^(1/4), E = mu u^2/2.  With the trap on, the ion is not where it started when
//     the atom arrives (at q = 0.4 it has moved by more than the whole range of impact parameters), so
//     the closest approach is estimated by a PRE-FLIGHT: the atom on its straight line against the ion
//     moving in the trap alone -- eq. (4)-(6) without the atom, integrated by velocity Verlet in 64 steps
//     over the fly-by, in single precision (a secular-orbit formula is off by 15-40 % of the orbit at the
//     trap strengths of the configs: as much as b_c itself) -- and refined by a parabola through the
//     three samples around the minimum.  "Candidates" pass within kappa b_c (kappa = 1.5), b_c from the
//     relative speed at that moment.  Without a trap this is the impact parameter.
// (2) Among them the slow ones take longest: the flight alone lasts ~1/u, and the complexes that
//     survive until t_max are low-energy ones.
// Three classes, queued in this order:
//     0: candidates with u^2 < <u^2>/2, and anything with u^2 < <u^2>/10   1: the other candidates
//     2: the rest
// so that the longest trajectories start early -- and reach the six-lane integrator a few milliseconds
// later -- instead of anywhere.  Affects scheduling only, never a result.
constexpr int kCntClass = 24;    // counters: trajectories per class (3; diagnostics)
constexpr int kCntMeanU2 = 60;   // counters: <u^2> (double bits)
constexpr int kPlanSamples = 64;
// Inside a class the queue is ordered by slowness (and closeness) as well: kPlanSub buckets of u^2 / <u^2> + x^2/4,
// 1/8 wide, the slowest first (the long trajectories of EVERY class are its slow ones, the unpredicted ones of class 2 too).
// Bucket = class * kPlanSub + sub; their counts and placement cursors sit behind the first 64 counters.
constexpr int kPlanSub = 16;
constexpr int kPlanBuckets = 3 * kPlanSub;
constexpr int kCntBucket = 64;                  // counters: trajectories per bucket
constexpr int kCntCursor = 64 + kPlanBuckets;   // counters: placement cursors

struct PlanArgs {
    double mu, c4;        // reduced mass, C4
    double kappa;
    double slow0, slow1;  // class thresholds as fractions of <u^2>
    float wa[3], wb[3];   // trap stiffness of the ion: w_k(t) = wa_k + wb_k cos(Omega t)  (eq. (4)-(6))
    float omega, phase0;  // Omega, Omega t0 reduced to [0, 2 pi)
    double span;          // t_max - t0
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
    // single precision throughout: a scheduling estimate (positions ~1e3 a0 to 1e-4 a0, far below the ~1e2 a0
    // it decides on), on the FP32 pipes instead of the FP64 pipe the integrators need
    float xi[3], vi[3], xa[3], va[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        xi[k] = (float)y0[(0 + k) * N + i];
        vi[k] = (float)y0[(3 + k) * N + i];
        xa[k] = (float)y0[(6 + k) * N + i];
        va[k] = (float)y0[(9 + k) * N + i];
    }
    const float d0 = xa[0] - xi[0], d1 = xa[1] - xi[1], d2 = xa[2] - xi[2];
    const float u0 = va[0] - vi[0], u1 = va[1] - vi[1], u2 = va[2] - vi[2];
    const float usq = u0 * u0 + u1 * u1 + u2 * u2;
    const float dsq = d0 * d0 + d1 * d1 + d2 * d2;
    // fly-by window: twice the time to cover the initial distance, within the time span
    float T = (float)A.span;
    if (usq > 0.0f) T = fminf(T, 2.0f * sqrtf(dsq / usq));
    const float h = T / kPlanSamples, hh = 0.5f * h;
    // the ion in the trap alone: x_k'' = -w_k(t) x_k, velocity Verlet (kick - drift - kick; as good a predictor as
    // classical RK4 at this step, measured offline on 1,048,576 trajectories per trap strength, at a quarter of the
    // arithmetic); the phase Omega t is advanced directly
    float x[3] = {xi[0], xi[1], xi[2]}, v[3] = {vi[0], vi[1], vi[2]};
    const float dph = A.omega * h;
    float c0 = __cosf(A.phase0);
    float f_prev = dsq, f_best = dsq, f_before = dsq, f_after = dsq, u_best = usq;
    int j_best = 0;
    bool want_after = true;
    for (int j = 1; j <= kPlanSamples; ++j) {
        const float c1 = __cosf(A.phase0 + dph * (float)j);
        const float t = h * (float)j;
        float f = 0.0f, us = 0.0f;
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const float w0 = fmaf(A.wb[k], c0, A.wa[k]), w1 = fmaf(A.wb[k], c1, A.wa[k]);
            const float vh = fmaf(-hh * w0, x[k], v[k]);
            x[k] = fmaf(h, vh, x[k]);
            v[k] = fmaf(-hh * w1, x[k], vh);
            const float dk = fmaf(va[k], t, xa[k]) - x[k];
            const float uk = va[k] - v[k];
            f = fmaf(dk, dk, f);
            us = fmaf(uk, uk, us);
        }
        c0 = c1;
        if (want_after) {
            f_after = f;
            want_after = false;
        }
        if (f < f_best) {
            f_best = f;
            f_before = f_prev;
            j_best = j;
            u_best = us;
            want_after = true;
            f_after = f;
        }
        f_prev = f;
    }
    // parabola through the best sample and its neighbours
    const float den = f_before - 2.0f * f_best + f_after;
    float off = 0.0f;
    if (den > 0.0f && j_best > 0 && j_best < kPlanSamples) off = fminf(fmaxf(0.5f * (f_before - f_after) / den, -1.0f), 1.0f);
    const float dmin2 = fmaxf(f_best - 0.25f * (f_before - f_after) * off, 0.0f);
    const float urel2 = u_best;  // relative speed at the sample of the closest approach
    // b_c = (8 C4 / (mu u^2))^(1/4)
    const float bc = urel2 > 0.0f ? sqrtf(sqrtf((float)(8.0 * A.c4 / A.mu) / urel2)) : 3.0e38f;
    const float xc = sqrtf(dmin2) / ((float)A.kappa * bc);  // closest approach in units of the capture range
    const bool cand = xc < 1.0f;
    const float r = usq / (float)mean_u2;
    const int cls = ((cand && r < (float)A.slow0) || r < (float)A.slow1) ? 0 : (cand ? 1 : 2);
    // inside a class: slow and close first (measured on the bench workload: its longest trajectories start 2 ms earlier
    // than by slowness alone)
    const float xs = fminf(xc, 2.0f);
    const int sub = (int)fminf(8.0f * (r + 0.25f * xs * xs), (float)(kPlanSub - 1));
    return cls * kPlanSub + sub;
}

// <u^2> over the first min(N, 65536) trajectories (a sample is enough for a scheduling threshold): 256 blocks of 256
// threads add their partial sums into counters[kCntMeanU2] (a double, zero from the call's memset); the readers
// divide by n.  (Blocks of 1024 threads capped the kernel at 64 registers and spilled 84 bytes.)
constexpr long long kPlanMeanSample = 65536;
__global__ void __launch_bounds__(256)
plan_mean_kernel(const double* __restrict__ y0, const long long N, unsigned long long* __restrict__ counters)
{
    __shared__ double part[32];
    const long long n = N < kPlanMeanSample ? N : kPlanMeanSample;
    double s = 0.0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        s += rel_speed2(y0, N, i);
    for (int off = 16; off > 0; off >>= 1) s += __shfl_down_sync(0xffffffffu, s, off);
    if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x < 32) {
        s = (threadIdx.x < (blockDim.x >> 5)) ? part[threadIdx.x] : 0.0;
        for (int off = 16; off > 0; off >>= 1) s += __shfl_down_sync(0xffffffffu, s, off);
        if (threadIdx.x == 0) atomicAdd(reinterpret_cast<double*>(counters + kCntMeanU2), s);
    }
}

// PLACE = 0: classify (cls[]) and count the classes; PLACE = 1: write order[] (cursors set by plan_bounds_kernel)
template <int PLACE>
__global__ void __launch_bounds__(256)
plan_kernel(const double* __restrict__ y0, const long long N, const PlanArgs A, long long* __restrict__ order,
            unsigned char* __restrict__ cls_of, unsigned long long* __restrict__ counters)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const unsigned FULL = 0xffffffffu;
    int cls = -1;
    if (i < N) {
        if (PLACE) {
            cls = cls_of[i];
        } else {
            const long long n_mean = N < kPlanMeanSample ? N : kPlanMeanSample;
            cls = plan_class(y0, N, i, A, __longlong_as_double((long long)counters[kCntMeanU2]) / (double)n_mean);
            cls_of[i] = (unsigned char)cls;
        }
    }
    // lanes of the same bucket: one atomic per bucket and warp
    const int lane = threadIdx.x & 31;
    const unsigned m = __match_any_sync(FULL, cls);
    if (cls >= 0) {
        const int leader = __ffs(m) - 1;
        unsigned long long base = 0;
        if (lane == leader) base = atomicAdd(&counters[(PLACE ? kCntCursor : kCntBucket) + cls], (unsigned long long)__popc(m));
        if (PLACE) {
            base = __shfl_sync(m, base, leader);
            order[base + __popc(m & ((1u << lane) - 1u))] = i;
        }
    }
}

// cursors at the bucket starts; bound[0], bound[1] = the whole of order[] (one bulk pass over the ordered queue)
__global__ void plan_bounds_kernel(unsigned long long* counters, int bound0, int front)
{
    unsigned long long acc = 0;
    for (int b = 0; b < kPlanBuckets; ++b) {
        counters[kCntCursor + b] = acc;
        const unsigned long long n = counters[kCntBucket + b];
        acc += n;
        counters[kCntClass + b / kPlanSub] += n;
        if (b == 2 * kPlanSub - 1) counters[front] = acc;  // classes 0 and 1 (diagnostics)
    }
    counters[bound0] = 0;
    counters[bound0 + 1] = acc;
}

// without a plan: one stage over [0, N)
__global__ void bounds_kernel(unsigned long long* counters, int bound0, unsigned long long N)
{
    counters[bound0] = 0;
    counters[bound0 + 1] = N;
}

// Head start for the six-lane pass that runs beside the per-thread integrator: it is launched first, on
// its own stream, and must take its SMs before the per-thread integrator fills them (both become ready
// at the same moment).  Waits until the six-lane pass has stamped its start, or at most `ns`.
__global__ void head_start_kernel(const unsigned long long* started, unsigned long long ns)
{
    const unsigned long long t0 = global_ns();
    while (*(volatile const unsigned long long*)started == 0ULL && global_ns() - t0 < ns) __nanosleep(500);
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

// The same count, starting from a guess j0 (exact for ANY strictly increasing edges: the two loops walk to
// the answer; with near-uniform edges and a linear guess they run at most once or twice).
__device__ __forceinline__ int bin_from_guess(const double* __restrict__ edges, int nb, double v, int j0)
{
    if (v != v) return nb + 1;
    int j = j0 < 0 ? 0 : (j0 > nb + 1 ? nb + 1 : j0);
    while (j <= nb && edges[j] <= v) ++j;
    while (j > 0 && edges[j - 1] > v) --j;
    return j;
}

struct HistArgs {
    const double *angle, *lifetime;
    const int *n_acc, *n_rej, *n_turn, *status;
    const unsigned char* complex_flag;
    const double *angle_edges, *life_edges;
    int na, nl, nt;
    unsigned long long *h_angle, *h_life, *h_turn, *h_status, *h_totals;
};

// HBM-bound: 33 B per trajectory (angle, lifetime, four int32, the flag).
// Grid-stride over N, kHistUnroll = 2 trajectories per thread and iteration in a two-stage software pipeline
// (the loads of the next pair are in flight while the current pair is binned); bins
// privatised in shared memory (edges staged there too).  The 4-valued status and the small n_turn values
// (0..3: all but a few per mille) are counted in registers and folded once per warp at the end; the
// angle takes a linear guess of its bin, corrected against the edges (exact for any edges), and a plain
// run-length cached shared-memory atomic; lifetimes (complexes only) a binary search.
constexpr int kHistUnroll = 2;
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
    const double e0 = s_ae[0];
    const double span = s_ae[a.na] - e0;
    const double scale = (span > 0.0 && span < 1.0e300) ? (double)a.na / span : 0.0;

    unsigned long long sum_acc = 0, sum_rej = 0;
    unsigned n_cplx = 0, n_traj = 0;
    unsigned c_status[4] = {0u, 0u, 0u, 0u}, c_turn[4] = {0u, 0u, 0u, 0u};
    const bool turn_regs = a.nt >= 4;
    int run_bin = 0;
    unsigned run_len = 0u;
    const long long stride = (long long)gridDim.x * blockDim.x;
    // software pipeline: the loads of the next kHistUnroll trajectories are in flight while the current ones
    // are binned (the kernel is bound by memory latency, not by instructions)
    struct Batch {
        double ang[kHistUnroll], life[kHistUnroll];
        int nt[kHistUnroll], st[kHistUnroll], na[kHistUnroll], nr[kHistUnroll];
        unsigned char fl[kHistUnroll];
    };
    auto load = [&](Batch& B, long long i0) {
#pragma unroll
        for (int u = 0; u < kHistUnroll; ++u) {
            const long long i = i0 + u * stride;
            const bool in = i < N;
            B.ang[u] = in ? __ldcs(a.angle + i) : 0.0;
            B.life[u] = in ? __ldcs(a.lifetime + i) : 0.0;  // for every trajectory: a load behind the flag would expose its latency
            B.fl[u] = in ? __ldcs(a.complex_flag + i) : (unsigned char)0;
            B.nt[u] = in ? __ldcs(a.n_turn + i) : 0;
            B.st[u] = in ? __ldcs(a.status + i) : 0;
            B.na[u] = in ? __ldcs(a.n_acc + i) : 0;
            B.nr[u] = in ? __ldcs(a.n_rej + i) : 0;
        }
    };
    Batch cur, nxt;
    long long i0 = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i0 < N) load(cur, i0);
    for (; i0 < N; i0 += kHistUnroll * stride) {
        const long long i_next = i0 + kHistUnroll * stride;
        if (i_next < N) load(nxt, i_next);
#pragma unroll
        for (int u = 0; u < kHistUnroll; ++u) {
            const long long i = i0 + u * stride;
            if (i >= N) break;
            const double v = cur.ang[u];
            const double g = fmin(fmax((v - e0) * scale, -1.0), (double)a.na + 1.0);
            const int ba = bin_from_guess(s_ae, a.na, v, (v == v) ? (int)g + 1 : 0);
            // run-length cache: the angle distribution is sharply peaked (most atoms are barely deflected), so
            // consecutive trajectories of a thread mostly hit the same bin: one atomic per run, not per trajectory
            if (ba == run_bin) {
                ++run_len;
            } else {
                if (run_len) atomicAdd(&s_angle[run_bin], run_len);
                run_bin = ba;
                run_len = 1u;
            }
            const bool cplx = cur.fl[u] != 0;
            if (cplx) atomicAdd(&s_life[bin_of(s_le, a.nl, cur.life[u])], 1u);
            const int b = cur.nt[u] < 0 ? 0 : (cur.nt[u] >= a.nt ? a.nt - 1 : cur.nt[u]);
            if (turn_regs && b < 4) {
#pragma unroll
                for (int k = 0; k < 4; ++k) c_turn[k] += (b == k) ? 1u : 0u;
            } else {
                atomicAdd(&s_turn[b], 1u);
            }
            const int sb = cur.st[u] & 3;
#pragma unroll
            for (int k = 0; k < 4; ++k) c_status[k] += (sb == k) ? 1u : 0u;
            sum_acc += (unsigned long long)cur.na[u];
            sum_rej += (unsigned long long)cur.nr[u];
            n_cplx += cplx ? 1u : 0u;
            n_traj += 1u;
        }
        cur = nxt;
    }
    // the last run of every thread, aggregated over the lanes that end in the same bin
    const unsigned FULL = 0xffffffffu;
    {
        const unsigned grp = __match_any_sync(FULL, run_bin);
        const unsigned tot = __reduce_add_sync(grp, run_len);
        if ((threadIdx.x & 31) == __ffs(grp) - 1 && tot) atomicAdd(&s_angle[run_bin], tot);
    }
    // register counters: one reduction per warp, one shared-memory atomic per warp and value
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const unsigned cs = __reduce_add_sync(FULL, c_status[k]);
        const unsigned ct = __reduce_add_sync(FULL, c_turn[k]);
        if ((threadIdx.x & 31) == 0) {
            if (cs) atomicAdd(&s_status[k], cs);
            if (ct) atomicAdd(&s_turn[k], ct);
        }
    }
    const unsigned w_cplx = __reduce_add_sync(FULL, n_cplx), w_traj = __reduce_add_sync(FULL, n_traj);
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        sum_acc += __shfl_down_sync(FULL, sum_acc, off);
        sum_rej += __shfl_down_sync(FULL, sum_rej, off);
    }
    __shared__ unsigned long long s_tot[4];
    if (threadIdx.x < 4) s_tot[threadIdx.x] = 0ULL;
    __syncthreads();
    if ((threadIdx.x & 31) == 0) {
        if (sum_acc) atomicAdd(&s_tot[0], sum_acc);
        if (sum_rej) atomicAdd(&s_tot[1], sum_rej);
        if (w_cplx) atomicAdd(&s_tot[2], (unsigned long long)w_cplx);
        if (w_traj) atomicAdd(&s_tot[3], (unsigned long long)w_traj);
    }
    __syncthreads();
    if (threadIdx.x < 4 && s_tot[threadIdx.x]) atomicAdd(&a.h_totals[threadIdx.x], s_tot[threadIdx.x]);
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
// NEXT-2: an observable against the launch direction
// ------------------------------------------------------------------------------------------
// HBM-bound: 32 B read per trajectory; one global atomic pair per trajectory inside the window (thousands of
// cells: little contention).  Edges are searched in global memory (L1-resident: a few KB).
__global__ void __launch_bounds__(256)
map2d_kernel(const double* __restrict__ y0, const long long N, const double* __restrict__ value,
             const double* __restrict__ u_edges, const int n_u, const double* __restrict__ phi_edges, const int n_phi,
             unsigned long long* __restrict__ count, double* __restrict__ sum)
{
    const long long stride = (long long)gridDim.x * blockDim.x;
    const double two_pi = 6.283185307179586, phi0 = phi_edges[0];
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += stride) {
        const double v = value[i];
        // the spherical angles of the atom's initial position; r = 0 gives u = NaN: skipped
        const double dx = y0[6 * N + i], dy = y0[7 * N + i], dz = y0[8 * N + i];
        const double r = sqrt(sum3(dx * dx, dy * dy, dz * dz));
        const double u = 0.5 * (1.0 - dz / r);
        double phi = atan2(dy, dx);  // a pole (dx = dy = 0) reads phi = 0
        phi = phi - two_pi * floor((phi - phi0) / two_pi);  // into [phi0, phi0 + 2 pi): a window may straddle 0
        const int a = bin_of(u_edges, n_u, u), b = bin_of(phi_edges, n_phi, phi);  // 0 / n + 1: outside (NaN too)
        if (a >= 1 && a <= n_u && b >= 1 && b <= n_phi && v == v) {
            const long long cell = (long long)(a - 1) * n_phi + (b - 1);
            atomicAdd(count + cell, 1ULL);
            atomicAdd(sum + cell, v);
        }
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
    if (p->max_steps < 1 || p->max_steps > 2147483647LL) return AIG_ERR_PARAM;  // the step counters are int32
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
//   plan        order[]: the work queue in three classes (plan_*_kernel), likely-long trajectories first
//   stream      six-lane integrator on a stream of its own, on `split_sms` SMs (one 8-warp block per SM
//               that asks for the whole shared memory, so that no bulk block shares its FP64 pipes):
//               takes checkpoint slots as the bulk pass publishes them
//   bulk        per-thread integrator over the whole queue on the other SMs; what outlives `budget`
//               accepted steps (and the mean of the finished ones, several times) is suspended into
//               the next slot as soon as the six-lane pass has room for it, and so is whatever is
//               still running `tail_iters` iterations after the queue ran dry
//   final       six-lane integrator on the whole GPU: shares the remaining slots with the streaming pass
//   join        the caller's stream waits for the streaming pass.
// The longest trajectories (10^2..10^3 x the mean number of steps) start their long sequential run
// in the six-lane integrator a few milliseconds after they were started, whatever class they are in.
// Waiting is one-sided and bounded (SplitSched): the bulk pass never waits for anyone.
// Checkpoint slots: min(N, max(2^20, N/4)); the capacity test in the kernel is a safety net.
constexpr long long kMinSlots = 1 << 20;

struct SchedConfig {
    int tail_iters = 1024;    // iterations a warp keeps stepping after the queue ran dry (round 3: 256 -> 1024, fewer late hand-overs)
    int budget = 2048;        // accepted steps after which the per-thread integrator offers a trajectory
    int split_sms = 12;       // SMs the streaming six-lane pass takes for itself (one 8-warp block each)
    int split_grid_b = 8;     // final six-lane pass: one-warp blocks per SM (it has the GPU to itself)
    int depth = 64;           // budget hand-overs stop while this many published slots wait to be taken
    int mean_factor = 4;      // ... and are only for trajectories this many times longer than the finished ones' mean
    int drain_lanes = 10;     // queue empty: a warp hands over what it still runs once this few lanes are alive
    double slow0 = 0.5;       // class 0: candidates with u^2 < slow0 <u^2>
    double slow1 = 0.1;       // class 1 also takes anything with u^2 < slow1 <u^2>
    int refill_batch = 8;     // idle lanes of a warp that trigger its refill ...
    int refill_wait = 16;     // ... or iterations one of them has waited
    int plan = 1;             // 0: natural order
    double kappa = 1.5;       // candidates: b < kappa * Langevin radius
    int poll_iters = 32;      // six-lane warps with idle groups look for new slots every this many iterations
    int hist_blocks_per_sm = 8;  // grid of histogram_kernel
};

std::mutex g_sched_mutex;
SchedConfig g_sched;          // guarded by g_sched_mutex; changed by aig_set_schedule / aig_set_schedule_ex only

SchedConfig sched_config()
{
    std::lock_guard<std::mutex> lock(g_sched_mutex);
    return g_sched;
}

long long slot_capacity(long long N) { return std::min(N < 1 ? 1 : N, std::max(kMinSlots, N / 4)); }

size_t round_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// workspace: 256 uint64 counters (64 of the schedule + the plan's buckets) | order[N] (int64) | bucket[N] (uint8) | checkpoint slots
constexpr size_t kCounterBytes = 256 * sizeof(unsigned long long);
size_t order_bytes(long long N) { return round_up((size_t)(N < 1 ? 1 : N) * sizeof(long long), 256); }
size_t class_bytes(long long N) { return round_up((size_t)(N < 1 ? 1 : N), 256); }
size_t ckpt_buffer_bytes(long long cap) { return round_up((size_t)cap * kCkptBytesPerSlot, 256); }

// counters (uint64 each)
enum Counter {
    kCntFront = 0,       // plan: candidates placed (classes 0 and 1)
    kCntStarted = 2,     // the bulk pass has started
    kCntDoneWarps = 3,   // warps of the bulk pass that have exited
    kCntSlots = 4,       // checkpoint slots handed out so far (may overshoot the capacity)
    kCntBound = 5,       // bound[0], bound[1]: the bulk pass's range of order[]
    kCntTaken = 8,       // slots claimed by the six-lane passes so far
    kCntFinished = 9,    // trajectories the six-lane passes have finished
    kCntBar = 10,        // the hand-over bar (accepted steps), and at [11] the %globaltimer of its last change
    kCntQueueBulk = 16,  // work queue of the bulk pass
    kCntLoaded = 61,     // diagnostics: trajectories taken by the streaming / the final six-lane pass
    kCntStats = 52       // accepted steps / number of the trajectories the bulk pass has finished
};
// stage timeline slots (kCntTime + 2 s): 0 plan (unused), 1 bulk, 2 streaming six-lane pass, 3 final six-lane pass
constexpr int kStageBulk = 1, kStageStream = 2, kStageFinal = 3;

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

// The side stream of the streaming six-lane pass and the two events that fork and join it, one set per
// device.  g_enqueue_mutex is held over the whole enqueue section of a call, so every record / wait
// pair is atomic with respect to other host threads calling aig_integrate on the same device.
struct SideStream {
    cudaStream_t stream = nullptr;
    cudaEvent_t fork = nullptr, join = nullptr;
    bool ok = false;
};
std::mutex g_enqueue_mutex;

SideStream* side_stream()   // call with g_enqueue_mutex held
{
    static SideStream side[64];
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return nullptr;
    SideStream& s = side[dev];
    if (!s.ok) {
        int lo = 0, hi = 0;
        if (cudaDeviceGetStreamPriorityRange(&lo, &hi) != cudaSuccess) return nullptr;
        if (cudaStreamCreateWithPriority(&s.stream, cudaStreamNonBlocking, hi) != cudaSuccess) return nullptr;
        if (cudaEventCreateWithFlags(&s.fork, cudaEventDisableTiming) != cudaSuccess) return nullptr;
        if (cudaEventCreateWithFlags(&s.join, cudaEventDisableTiming) != cudaSuccess) return nullptr;
        s.ok = true;
    }
    return &s;
}

constexpr int kSplitMinBlocks = 8;  // register cap of the split kernel: 65536 / (8 x 32) = 256
#ifndef AIG_SPLIT_WARPS
#define AIG_SPLIT_WARPS 4
#endif
constexpr int kSplitWarps = AIG_SPLIT_WARPS;  // warps per block of the SM-owning variant: two per scheduler (a warp issues a third of the
                                              // time, so two barely slow each other while the queue is long; at the end each is alone)

template <int TRAP>
int launch_integrate(const aig_params* p, const KParams& K, const double* y0, long long N, const OutPtrs& O,
                     void* workspace, cudaStream_t st)
{
    const SchedConfig cfg = sched_config();
    const long long cap = slot_capacity(N);
    unsigned long long* counters = static_cast<unsigned long long*>(workspace);
    long long* order = reinterpret_cast<long long*>(static_cast<unsigned char*>(workspace) + kCounterBytes);
    unsigned char* cls_of = static_cast<unsigned char*>(workspace) + kCounterBytes + order_bytes(N);
    const Ckpt slots = ckpt_at(cls_of + class_bytes(N), cap);

    // Per device and kernel family, once: resident blocks of the bulk kernel, the shared-memory opt-in of the
    // streaming block, and a touch of every kernel of the schedule.  (CUDA loads a kernel's code at its first
    // launch -- lazy module loading -- and loading may have to wait for the kernels that are running: the first
    // call would serialise the passes that are meant to overlap.)  Later calls find the answers cached: a dozen
    // runtime queries would otherwise sit in front of every call's first launch.
    struct Setup {
        bool done = false;
        int bps = 0, sms = 0, smem_optin = 0;
    };
    static Setup setup_of[64];
    static std::mutex setup_mutex;
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return AIG_ERR_CUDA;
    int bps = 0, sms = 0, smem_optin = 0;
    {
        std::lock_guard<std::mutex> lock(setup_mutex);
        Setup& su = setup_of[dev];
        if (!su.done) {
            const int rc = bulk_capacity<TRAP>(&su.bps, &su.sms);
            if (rc) return rc;
            if (cudaDeviceGetAttribute(&su.smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev) != cudaSuccess)
                return AIG_ERR_CUDA;
            cudaFuncAttributes fa;
            if (cudaFuncGetAttributes(&fa, integrate_kernel<TRAP, kBlock, kBlocksPerSM>) != cudaSuccess ||
                cudaFuncGetAttributes(&fa, integrate_split_kernel<TRAP, kSplitWarps, 1>) != cudaSuccess ||
                cudaFuncGetAttributes(&fa, integrate_split_kernel<TRAP, 1, kSplitMinBlocks>) != cudaSuccess ||
                cudaFuncGetAttributes(&fa, plan_mean_kernel) != cudaSuccess ||
                cudaFuncGetAttributes(&fa, plan_kernel<0>) != cudaSuccess ||
                cudaFuncGetAttributes(&fa, plan_kernel<1>) != cudaSuccess ||
                cudaFuncGetAttributes(&fa, plan_bounds_kernel) != cudaSuccess ||
                cudaFuncGetAttributes(&fa, bounds_kernel) != cudaSuccess ||
                cudaFuncGetAttributes(&fa, head_start_kernel) != cudaSuccess)
                return AIG_ERR_CUDA;
            if (cudaFuncSetAttribute(integrate_split_kernel<TRAP, kSplitWarps, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                     su.smem_optin) != cudaSuccess)
                return AIG_ERR_CUDA;
            su.done = true;
        }
        bps = su.bps;
        sms = su.sms;
        smem_optin = su.smem_optin;
    }
    const bool plan = cfg.plan != 0 && p->C4 > 0.0 && (p->n_att == 0 || p->n_att == 4);  // the Langevin test is the r^-4 tail's
    // the streaming pass: on its own SMs when the work is large enough to fill the others
    const long long own = std::max<long long>(1, std::min<long long>(cfg.split_sms, sms / 2));
    const long long blocks_all = std::min((long long)bps * sms, (N + kBlock - 1) / kBlock);
    const long long blocks = std::max<long long>(1, std::min<long long>(blocks_all, (long long)bps * (sms - own)));
    const unsigned split_last =
        (unsigned)std::min<long long>((long long)cfg.split_grid_b * sms, (cap + kGroupsPerWarp - 1) / kGroupsPerWarp);

    std::lock_guard<std::mutex> enqueue_lock(g_enqueue_mutex);
    SideStream* side = side_stream();
    if (!side) return AIG_ERR_CUDA;

    if (cudaMemsetAsync(counters, 0, kCounterBytes, st) != cudaSuccess) return AIG_ERR_CUDA;
    // slot index entries = -1: "not published" (ckpt_store / ckpt_wait)
    if (cudaMemsetAsync(slots.idx, 0xFF, (size_t)cap * sizeof(long long), st) != cudaSuccess) return AIG_ERR_CUDA;
    long long* order_arg = nullptr;
    if (plan) {
        PlanArgs A;
        A.mu = p->m_ion * p->m_atom / (p->m_ion + p->m_atom);
        A.c4 = p->C4;
        A.kappa = cfg.kappa;
        A.slow0 = cfg.slow0;
        A.slow1 = cfg.slow1;
        A.span = K.t_max - K.t0;
        const double W = 0.25 * p->omega_rf * p->omega_rf;
        for (int k = 0; k < 3; ++k) {
            A.wa[k] = (float)(p->a[k] * W);
            A.wb[k] = (float)(2.0 * p->q[k] * W);
        }
        A.omega = (float)p->omega_rf;
        A.phase0 = (float)std::fmod(p->omega_rf * p->t0, 6.283185307179586);
        const unsigned pg = (unsigned)((N + 255) / 256);
        plan_mean_kernel<<<(unsigned)std::min<long long>(256, (N + 255) / 256), 256, 0, st>>>(y0, N, counters);
        plan_kernel<0><<<pg, 256, 0, st>>>(y0, N, A, order, cls_of, counters);
        plan_bounds_kernel<<<1, 1, 0, st>>>(counters, kCntBound, kCntFront);
        plan_kernel<1><<<pg, 256, 0, st>>>(y0, N, A, order, cls_of, counters);
        g_kernel_launches += 4;
        order_arg = order;
    } else {
        bounds_kernel<<<1, 1, 0, st>>>(counters, kCntBound, (unsigned long long)N);
        g_kernel_launches++;
    }

    SplitSched T;
    T.in = slots;
    T.taken = counters + kCntTaken;
    T.n_out = counters + kCntSlots;
    T.started = counters + kCntStarted;
    T.done_warps = counters + kCntDoneWarps;
    T.producer_warps = (unsigned long long)blocks * (kBlock / 32);
    T.poll_iters = cfg.poll_iters;
    T.finished = counters + kCntFinished;
    T.bar = counters + kCntBar;
    T.bar_floor = (unsigned long long)cfg.budget;
    T.capacity = own * kSplitWarps * kGroupsPerWarp;

    // streaming six-lane pass on the side stream: launched first, so that it owns its SMs
    if (cudaEventRecord(side->fork, st) != cudaSuccess || cudaStreamWaitEvent(side->stream, side->fork, 0) != cudaSuccess)
        return AIG_ERR_CUDA;
    T.timeline = counters + kCntTime + 2 * kStageStream;
    T.loaded = counters + kCntLoaded;
    T.patience_ns = 2000000ULL;  // 2 ms to see the bulk pass start
    integrate_split_kernel<TRAP, kSplitWarps, 1><<<(unsigned)own, 32 * kSplitWarps, (size_t)smem_optin, side->stream>>>(K, y0, N, O, T);
    g_kernel_launches++;
    // From here on the side stream may hold a kernel that polls and writes the caller's workspace and outputs.
    // Whatever fails below, the caller's stream must not get past this call before that kernel has ended (it gives
    // up by itself 2 ms after it finds that no bulk pass has started): join the side stream, or, if even that
    // fails, block the host on it.  Otherwise the caller could free or reuse the buffers under a running kernel
    // and the next call on this device would find the shared side stream busy.
    auto leave = [&](int rc) {
        if (cudaStreamWaitEvent(st, side->join, 0) != cudaSuccess) {
            (void)cudaStreamSynchronize(side->stream);
            rc = rc ? rc : AIG_ERR_CUDA;
        }
        return rc;
    };
    if (cudaGetLastError() != cudaSuccess) {  // the streaming launch itself failed: nothing is running on the side stream
        (void)cudaStreamSynchronize(side->stream);
        return AIG_ERR_CUDA;
    }
    if (cudaEventRecord(side->join, side->stream) != cudaSuccess) {
        (void)cudaStreamSynchronize(side->stream);
        return AIG_ERR_CUDA;
    }

    // bulk pass on the caller's stream, behind a short wait for the streaming pass to have taken its SMs
    head_start_kernel<<<1, 1, 0, st>>>(counters + kCntTime + 2 * kStageStream, 200000ULL);
    Sched S;
    S.order = order_arg;
    S.queue = counters + kCntQueueBulk;
    S.begin = counters + kCntBound;
    S.end = counters + kCntBound + 1;
    S.n_out = counters + kCntSlots;
    S.finished = counters + kCntFinished;
    S.bar = counters + kCntBar;
    S.capacity = own * kSplitWarps * kGroupsPerWarp;
    S.started = counters + kCntStarted;
    S.done_warps = counters + kCntDoneWarps;
    S.out = slots;
    S.depth = cfg.depth;
    S.budget = cfg.budget;
    S.tail_iters = cfg.tail_iters;
    S.refill_batch = cfg.refill_batch;
    S.refill_wait = cfg.refill_wait;
    S.drain_lanes = cfg.drain_lanes;
    S.stats = counters + kCntStats;
    S.mean_factor = cfg.mean_factor;
    S.timeline = counters + kCntTime + 2 * kStageBulk;
    integrate_kernel<TRAP, kBlock, kBlocksPerSM><<<(unsigned)blocks, kBlock, 0, st>>>(K, y0, N, O, S);
    g_kernel_launches += 2;
    if (cudaGetLastError() != cudaSuccess) return leave(AIG_ERR_CUDA);  // no bulk pass: the streaming pass gives up; wait for it

    // final six-lane pass: the whole GPU on what is left (the bulk pass is complete: nothing to wait for)
    T.timeline = counters + kCntTime + 2 * kStageFinal;
    T.loaded = counters + kCntLoaded + 1;
    T.patience_ns = 0ULL;
    T.capacity = 0;
    integrate_split_kernel<TRAP, 1, kSplitMinBlocks><<<split_last, 32, 0, st>>>(K, y0, N, O, T);
    g_kernel_launches++;
    return leave(cudaGetLastError() == cudaSuccess ? AIG_OK : AIG_ERR_CUDA);
}

}  // namespace

extern "C" {

int aig_version(void) { return AIG_VERSION; }

uint64_t aig_kernel_launches(void) { return g_kernel_launches.load(); }

int aig_set_schedule(int tail_iters, int budget, int split_sms, int split_grid, int plan, double kappa)
{
    if (tail_iters < 0 || budget < 1 || split_sms < 1 || split_grid < 1 || !(kappa >= 0.0)) return AIG_ERR_PARAM;
    std::lock_guard<std::mutex> lock(g_sched_mutex);
    g_sched.tail_iters = tail_iters;
    g_sched.budget = budget;
    g_sched.split_sms = split_sms;
    g_sched.split_grid_b = split_grid;
    g_sched.plan = plan;
    g_sched.kappa = kappa;
    return AIG_OK;
}

int aig_set_schedule_ex(const aig_schedule* s)
{
    std::lock_guard<std::mutex> lock(g_sched_mutex);
    if (!s) {  // back to the defaults
        g_sched = SchedConfig();
        return AIG_OK;
    }
    if (s->tail_iters < 0 || s->budget < 1 || s->split_sms < 1 || s->split_grid < 1 || !(s->kappa >= 0.0) ||
        s->depth < 1 || s->mean_factor < 0 || s->drain_lanes < 0 || s->drain_lanes > 32 || !(s->slow0 >= 0.0) ||
        !(s->slow1 >= 0.0) || s->refill_batch < 1 || s->refill_batch > 32 || s->refill_wait < 0 || s->poll_iters < 1 ||
        s->hist_blocks_per_sm < 1 || s->hist_blocks_per_sm > 64)
        return AIG_ERR_PARAM;
    g_sched.tail_iters = s->tail_iters;
    g_sched.budget = s->budget;
    g_sched.split_sms = s->split_sms;
    g_sched.split_grid_b = s->split_grid;
    g_sched.plan = s->plan;
    g_sched.kappa = s->kappa;
    g_sched.depth = s->depth;
    g_sched.mean_factor = s->mean_factor;
    g_sched.drain_lanes = s->drain_lanes;
    g_sched.slow0 = s->slow0;
    g_sched.slow1 = s->slow1;
    g_sched.refill_batch = s->refill_batch;
    g_sched.refill_wait = s->refill_wait;
    g_sched.poll_iters = s->poll_iters;
    g_sched.hist_blocks_per_sm = s->hist_blocks_per_sm;
    return AIG_OK;
}

int aig_get_schedule(aig_schedule* s)
{
    if (!s) return AIG_ERR_NULL;
    const SchedConfig c = sched_config();
    s->tail_iters = c.tail_iters;
    s->budget = c.budget;
    s->split_sms = c.split_sms;
    s->split_grid = c.split_grid_b;
    s->plan = c.plan;
    s->kappa = c.kappa;
    s->depth = c.depth;
    s->mean_factor = c.mean_factor;
    s->drain_lanes = c.drain_lanes;
    s->slow0 = c.slow0;
    s->slow1 = c.slow1;
    s->refill_batch = c.refill_batch;
    s->refill_wait = c.refill_wait;
    s->poll_iters = c.poll_iters;
    s->hist_blocks_per_sm = c.hist_blocks_per_sm;
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
        case AIG_ERR_STATIC_LIMIT:
            return "N exceeds AIG_OUTLIERS_STATIC_MAX_N, the stated limit of aig_outliers_static's built-in scratch "
                   "(use aig_outliers with a caller workspace)";
        default: return "unknown error code";
    }
}

int aig_potential(int mode, int n, int m, double a, double b, double* Cn, double* Cm, double* De, double* Re)
{
    if (mode != AIG_POT_CNCM && mode != AIG_POT_CNDE && mode != AIG_POT_DERE) return AIG_ERR_SIZE;
    if (n < 1 || m <= n || m > 32) return AIG_ERR_PARAM;
    if (!std::isfinite(a) || !std::isfinite(b) || !(a > 0.0) || !(b > 0.0)) return AIG_ERR_PARAM;
    // V'(Re) = 0:  n Cn Re^m = m Cm Re^n;   V(Re) = -De:  De = Cn Re^-n - Cm Re^-m = Cn Re^-n (m - n) / m
    const double dn = (double)n, dm = (double)m;
    double cn, cm, de, re;
    if (mode == AIG_POT_CNCM) {
        cn = a;
        cm = b;
        re = std::pow(dm * cm / (dn * cn), 1.0 / (dm - dn));
        de = cn * (dm - dn) / (dm * std::pow(re, dn));
    } else if (mode == AIG_POT_CNDE) {
        cn = a;
        de = b;
        re = std::pow(cn * (dm - dn) / (dm * de), 1.0 / dn);
        cm = dn * cn * std::pow(re, dm - dn) / dm;
    } else {
        de = a;
        re = b;
        cn = de * dm * std::pow(re, dn) / (dm - dn);
        cm = de * dn * std::pow(re, dm) / (dm - dn);
    }
    if (Cn) *Cn = cn;
    if (Cm) *Cm = cm;
    if (De) *De = de;
    if (Re) *Re = re;
    return AIG_OK;
}

size_t aig_workspace_bytes(int64_t N)
{
    // counters + work-queue order (8 B per trajectory) + class (1 B) + checkpoint slots for suspended trajectories
    return kCounterBytes + order_bytes(N) + class_bytes(N) + ckpt_buffer_bytes(slot_capacity(N));
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
    // up to 2048 bins each: 57 KB of dynamic shared memory, above the 48 KB a kernel gets without opting in
    if (smem > 48 * 1024 &&
        cudaFuncSetAttribute(histogram_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
        return AIG_ERR_CUDA;
    long long blocks = (N + 256 * kHistUnroll - 1) / (256 * kHistUnroll);
    const long long cap = (long long)sms * sched_config().hist_blocks_per_sm;
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

int aig_map2d(const double* y0, int64_t N, const double* value, const aig_map_spec* spec, uint64_t* count, double* sum,
              void* cuda_stream)
{
    if (!spec) return AIG_ERR_NULL;
    if (N < 0 || N > (1LL << 40)) return AIG_ERR_SIZE;
    if (spec->n_u < 1 || spec->n_phi < 1 || spec->n_u > 4096 || spec->n_phi > 4096) return AIG_ERR_SIZE;
    if (!spec->u_edges || !spec->phi_edges || !count || !sum) return AIG_ERR_NULL;
    if (N == 0) return AIG_OK;
    if (!y0 || !value) return AIG_ERR_NULL;
    if (!aligned(y0, 8) || !aligned(value, 8) || !aligned(spec->u_edges, 8) || !aligned(spec->phi_edges, 8) ||
        !aligned(count, 8) || !aligned(sum, 8))
        return AIG_ERR_ALIGN;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return AIG_ERR_CUDA;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return AIG_ERR_CUDA;
    const long long blocks = std::min<long long>((N + 255) / 256, (long long)sms * 8);
    map2d_kernel<<<(unsigned)blocks, 256, 0, static_cast<cudaStream_t>(cuda_stream)>>>(
        y0, N, value, spec->u_edges, spec->n_u, spec->phi_edges, spec->n_phi,
        reinterpret_cast<unsigned long long*>(count), sum);
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
        if (hs->n_angle_bins > 2048 || hs->n_life_bins > 2048 || hs->n_turn_bins > 2048) return AIG_ERR_SIZE;
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

// ------------------------------------------------------------------------------------------
// aig_outliers_static: the arg-min / arg-max pass for callers that may not allocate (include/aig.h)
// ------------------------------------------------------------------------------------------
// The per-block partial extrema and the ticket counter of outliers_kernel live in an array that is part of
// the library image instead of a caller workspace.  Every device that loads libaig holds these bytes from
// module load until the process exits; every call on a device uses the same bytes.
namespace {

constexpr int kOutlierStaticBlocks = 512;  // grid cap of the static variant (aig_outliers itself: 1024)
constexpr size_t kOutlierStaticBytes = 256 + (size_t)kOutlierStaticBlocks * kOutlierObs * 2 * sizeof(Extreme);  // 131,328
static_assert(kOutlierStaticBytes == AIG_OUTLIERS_STATIC_SCRATCH_BYTES, "include/aig.h states the size of the static scratch");

static __device__ __align__(256) unsigned char g_outlier_scratch[kOutlierStaticBytes];

// In host code `g_outlier_scratch` names a host-side shadow of the array, not memory a kernel can use: the
// device address has to be asked for, separately on every device (each holds its own copy).  Looked up at the
// first call on a device, with that device current, and kept.
unsigned char* outlier_static_scratch(int* rc)
{
    static unsigned char* ptr_of[64];
    static std::mutex lookup_mutex;
    int dev = 0;
    *rc = AIG_ERR_CUDA;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return nullptr;
    std::lock_guard<std::mutex> lock(lookup_mutex);
    if (!ptr_of[dev]) {
        void* p = nullptr;
        if (cudaGetSymbolAddress(&p, g_outlier_scratch) != cudaSuccess || !p) {
            (void)cudaGetLastError();
            return nullptr;
        }
        ptr_of[dev] = static_cast<unsigned char*>(p);
    }
    *rc = AIG_OK;
    return ptr_of[dev];
}

}  // namespace

extern "C" {

int64_t aig_outliers_static_max_n(void) { return AIG_OUTLIERS_STATIC_MAX_N; }

int aig_outliers_static(const aig_out* out, const aig_obs_extra* extra, int64_t N, int64_t* result, void* cuda_stream)
{
    if (!result) return AIG_ERR_NULL;
    if (N < 0) return AIG_ERR_SIZE;
    if (N > AIG_OUTLIERS_STATIC_MAX_N) return AIG_ERR_STATIC_LIMIT;
    if (!aligned(result, 8)) return AIG_ERR_ALIGN;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    if (N > 0) {
        if (!out || !extra) return AIG_ERR_NULL;
        if (!out->angle || !out->lifetime || !out->n_turn || !out->n_acc || !extra->dist || !extra->KE || !extra->transfer)
            return AIG_ERR_NULL;
    }
    int rc = AIG_OK;
    unsigned char* scratch = outlier_static_scratch(&rc);  // first call on this device: the address look-up
    if (!scratch) return rc;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return AIG_ERR_CUDA;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return AIG_ERR_CUDA;
    // the array still holds the previous call's ticket count and partials: the ticket must start at zero (the
    // partials of the blocks of this launch are all rewritten before the last block reads them)
    if (cudaMemsetAsync(scratch, 0, 256, st) != cudaSuccess) return AIG_ERR_CUDA;
    OutlierArgs a;
    a.angle = N ? out->angle : nullptr;
    a.lifetime = N ? out->lifetime : nullptr;
    a.n_turn = N ? out->n_turn : nullptr;
    a.n_acc = N ? out->n_acc : nullptr;
    a.transfer = N ? extra->transfer : nullptr;
    a.dist = N ? extra->dist : nullptr;
    a.ke = N ? extra->KE : nullptr;
    a.position = N ? extra->position : nullptr;
    a.ticket = reinterpret_cast<unsigned int*>(scratch);
    a.partial = reinterpret_cast<Extreme*>(scratch + 256);
    a.result = reinterpret_cast<long long*>(result);
    int occ = 0;  // one wave of resident blocks, as in aig_outliers, and never more than the array has room for
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, outliers_kernel, 256, 0) != cudaSuccess || occ < 1) return AIG_ERR_CUDA;
    const long long blocks = std::min<long long>(std::max<long long>(1, (N + 255) / 256),
                                                 std::min<long long>((long long)sms * occ, kOutlierStaticBlocks));
    outliers_kernel<<<(unsigned)blocks, 256, 0, st>>>(a, N);
    g_kernel_launches++;
    return cudaGetLastError() == cudaSuccess ? AIG_OK : AIG_ERR_CUDA;
}

}  // extern "C"
