// aig_kernels.cu -- kernels and C ABI of libaig (include/aig.h).  sm_100a only.
//
// Kernels
//   integrate_kernel<TRAP> : persistent threads, one trajectory per lane, registers only;
//                            finished lanes refill from a global atomic work queue
//                            (warp-aggregated: one atomicAdd per warp per refill event).
//   step_once_kernel<TRAP> : test hook, one attempted step per thread.
//   histogram_kernel       : shared-memory privatised bins, warp-aggregated increments.
//   dfma_probe_kernel      : FP64 FMA chains, measures the non-tensor FP64 roofline.
//
// Nothing here is a dense contraction: no tensor cores, no TMA.  The bound is the FP64 pipe;
// global memory sees 96 B in and ~150 B out per trajectory against ~1e5 flops.
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <algorithm>
#include <atomic>
#include <cstdlib>
#include <cuda_runtime.h>

#include "../../include/aig.h"
#include "aig_device.cuh"

namespace aig {

#ifndef AIG_BLOCK
#define AIG_BLOCK 128
#endif
#ifndef AIG_MIN_BLOCKS
#define AIG_MIN_BLOCKS 2
#endif
constexpr int kBlock = AIG_BLOCK;             // threads per block of the integrator
constexpr int kBlocksPerSM = AIG_MIN_BLOCKS;  // resident blocks per SM the register budget is sized for

struct OutPtrs {
    double *y_final, *t_final, *lifetime, *angle, *r_min;
    int *n_acc, *n_rej, *n_turn, *status;
    unsigned char* complex_flag;
};

// ------------------------------------------------------------------------------------------
// integrator
// ------------------------------------------------------------------------------------------
// Cold state of the per-thread integrator: one shared-memory slot per thread, SoA (conflict-free).
struct ColdShared {
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

template <class Cold>
__device__ __forceinline__ void store_traj(const KParams& P, const double* __restrict__ y0,
                                           long long N, long long idx, const Traj& T, Cold& C, int status,
                                           const OutPtrs& O)
{
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        O.y_final[(0 + k) * N + idx] = T.X[k];
        O.y_final[(3 + k) * N + idx] = T.V[k];
        O.y_final[(6 + k) * N + idx] = T.X[3 + k];
        O.y_final[(9 + k) * N + idx] = T.V[3 + k];
    }
    O.t_final[idx] = T.t;
    const double v0[3] = {__ldg(y0 + 9 * N + idx), __ldg(y0 + 10 * N + idx), __ldg(y0 + 11 * N + idx)};
    const double v1[3] = {T.V[3], T.V[4], T.V[5]};
    O.angle[idx] = angle_between(v0, v1);
    O.r_min[idx] = sqrt(C.rmin2());
    const int n_turn = C.n_turn();
    const bool cplx = n_turn >= 2;
    O.lifetime[idx] = cplx ? C.t_last() - C.t_first() : 0.0;
    O.n_acc[idx] = T.n_acc;
    O.n_rej[idx] = C.n_rej();
    O.n_turn[idx] = n_turn;
    O.status[idx] = status;
    O.complex_flag[idx] = cplx ? 1 : 0;
}

// Checkpoint slots: the full state of a suspended trajectory, SoA over `cap` slots
// (d: 24 doubles per slot, i: 4 ints, idx: the trajectory's global index).
struct Ckpt {
    double* d;
    int* i;
    long long* idx;
    int cap;
};
constexpr int kCkptDoubles = 24, kCkptInts = 4;
constexpr size_t kCkptBytesPerSlot = kCkptDoubles * 8 + kCkptInts * 4 + 8;

template <class Cold>
__device__ __forceinline__ void ckpt_store(const Ckpt& K, int slot, long long idx, const Traj& T, Cold& C)
{
    double* d = K.d + slot;
    const size_t cap = (size_t)K.cap;
#pragma unroll
    for (int j = 0; j < 6; ++j) {
        d[(0 + j) * cap] = T.X[j];
        d[(6 + j) * cap] = T.V[j];
        d[(12 + j) * cap] = T.A1[j];
    }
    d[18 * cap] = T.t;
    d[19 * cap] = T.h;
    d[20 * cap] = T.sprev;
    d[21 * cap] = C.rmin2();
    d[22 * cap] = C.t_first();
    d[23 * cap] = C.t_last();
    int* q = K.i + slot;
    q[0 * cap] = T.n_acc;
    q[1 * cap] = (int)T.flags;
    q[2 * cap] = C.n_rej();
    q[3 * cap] = C.n_turn();
    K.idx[slot] = idx;
}

template <class Cold>
__device__ __forceinline__ long long ckpt_load(const Ckpt& K, int slot, Traj& T, Cold& C)
{
    const double* d = K.d + slot;
    const size_t cap = (size_t)K.cap;
#pragma unroll
    for (int j = 0; j < 6; ++j) {
        T.X[j] = d[(0 + j) * cap];
        T.V[j] = d[(6 + j) * cap];
        T.A1[j] = d[(12 + j) * cap];
    }
    T.t = d[18 * cap];
    T.h = d[19 * cap];
    T.sprev = d[20 * cap];
    C.rmin2() = d[21 * cap];
    C.t_first() = d[22 * cap];
    C.t_last() = d[23 * cap];
    const int* q = K.i + slot;
    T.n_acc = q[0 * cap];
    T.flags = (unsigned)q[1 * cap];
    C.n_rej() = q[2 * cap];
    C.n_turn() = q[3 * cap];
    return K.idx[slot];
}

// Scheduling arguments of one integrator launch (a stage of the schedule in aig_integrate).
//   fresh stage  (RESUME = 0): work items are trajectory indices [0, N), state from y0;
//   resume stage (RESUME = 1): work items are the slots [0, *n_in) of `in`, state from the slot.
// A lane whose trajectory has neither ended nor been suspended keeps stepping; it is suspended
// (state written to `out`, slot taken from *n_out) when it has taken `budget` accepted steps
// in this stage, or -- fresh stage only -- `tail_iters` iterations after its warp has seen the
// queue empty.  Suspension never changes a trajectory's arithmetic, only where it continues.
struct Sched {
    unsigned long long* queue;
    const unsigned long long* n_in;
    unsigned long long* n_out;
    Ckpt in, out;
    int budget;
    int tail_iters;
};

template <int TRAP, int RESUME, int BLOCK, int MINB>
__global__ void __launch_bounds__(BLOCK, MINB)
integrate_kernel(const KParams P, const double* __restrict__ y0, const long long N, const OutPtrs O,
                 const Sched S)
{
    __shared__ double s_rmin2[BLOCK], s_tfirst[BLOCK], s_tlast[BLOCK];
    __shared__ int s_nrej[BLOCK], s_nturn[BLOCK];
    ColdShared C{s_rmin2, s_tfirst, s_tlast, s_nrej, s_nturn};
    const unsigned FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    const long long total = RESUME ? (long long)*S.n_in : N;
    Traj T;
    long long idx = -1;
    int stop_at = 0;     // suspend when n_acc reaches this
    int since_dry = 0;   // warp-uniform: iterations since the queue was seen empty
    bool live = false;
    bool dry = false;    // warp-uniform: the queue has been seen empty

    for (;;) {
        // ---- refill: lanes without a trajectory take the next items of the queue
        const unsigned need = __ballot_sync(FULL, !live);
        if (need) {
            if (!dry) {
                const int cnt = __popc(need);
                const int leader = __ffs(need) - 1;
                unsigned long long base = 0;
                if (lane == leader) base = atomicAdd(S.queue, (unsigned long long)cnt);
                base = __shfl_sync(FULL, base, leader);
                if (!live) {
                    const long long cand = (long long)base + __popc(need & ((1u << lane) - 1u));
                    if (cand < total) {
                        if (RESUME) {
                            idx = ckpt_load(S.in, (int)cand, T, C);
                        } else {
                            idx = cand;
                            load_traj<TRAP>(P, y0, N, idx, T, C);
                        }
                        stop_at = (S.budget > 0x7fffffff - T.n_acc) ? 0x7fffffff : T.n_acc + S.budget;
                        live = true;
                    }
                }
                if ((long long)base + cnt >= total) dry = true;
            }
            if (!__any_sync(FULL, live)) break;
        }
        bool suspend = false;
        if (!RESUME && dry) suspend = (++since_dry > S.tail_iters);
        // ---- one attempted step for every live lane
        if (live) {
            if (!suspend) {
                Attempt R;
                dp45_attempt<TRAP>(P, T, R);
                const int st = finish_attempt(P, T, C, R);
                if (st >= 0) {
                    store_traj(P, y0, N, idx, T, C, st, O);
                    live = false;
                } else {
                    suspend = T.n_acc >= stop_at;
                }
            }
            if (live && suspend) {
                const int slot = (int)atomicAdd(S.n_out, 1ULL);
                ckpt_store(S.out, slot, idx, T, C);
                live = false;
            }
        }
    }
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
    T.t = t[i];
    T.h = h[i];
    T.flags = 0u;
    double r2;
    Attempt R;
    // RF trap: the branch-free cos where it is valid, libdevice's beyond (the integrator makes
    // this choice once per call on the host, from t0 and t_max)
    if (TRAP == TRAP_RF && !(fabs(P.omega) * (fabs(T.t) + fabs(T.h)) < 0.99 * kCosMaxArg)) {
        accel<TRAP_RF_BIG>(P, trap_cos<TRAP_RF_BIG>(P, T.t), T.X, T.A1, r2);
        dp45_attempt<TRAP_RF_BIG>(P, T, R);
    } else {
        accel<TRAP>(P, trap_cos<TRAP>(P, T.t), T.X, T.A1, r2);
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

KParams make_kparams(const aig_params* p, double t_max, double rtol, double atol)
{
    KParams K;
    K.inv_mi = 1.0 / p->m_ion;
    K.inv_ma = 1.0 / p->m_atom;
    K.c4x4 = 4.0 * p->C4;
    K.c8x8 = 8.0 * p->C8;
    const double w2 = p->omega_rf * p->omega_rf;
    for (int k = 0; k < 3; ++k) {
        K.wa[k] = p->a[k] * w2 / 4.0;
        K.wb[k] = p->q[k] * w2 / 2.0;
    }
    K.omega = p->omega_rf;
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
// Stage 0 (fresh): persistent grid of kBlock-thread blocks over the trajectory indices; lanes still
// running kTailIters iterations after their warp saw the queue empty are suspended into checkpoint
// buffer 0.  Stages 1..kRounds (resume): one-warp blocks over the slots the previous stage
// wrote, so the few long-lived trajectories (bound complexes take 10^2..10^3 times the mean number
// of steps) are packed densely into few warps spread over all SMs instead of idling 31 lanes of
// many warps that share a sub-partition's FP64 pipe; each round suspends what exceeds its step
// budget (x4 per round) into the other buffer, the last round has no budget.
constexpr int kRounds = 6;
constexpr int kRoundBlock = 32;
constexpr int kMaxSlots = 65536;  // checkpoint slots per buffer = upper bound on stage-0 lanes

struct SchedConfig {
    int tail_iters = 256;     // stage 0: iterations a warp keeps stepping after the queue ran dry
    int budget0 = 1 << 30;    // stage 0: accepted-step budget per trajectory (off)
    int round_budget = 1024;  // round 1 budget; x4 per round; the last round is unbounded
    int rounds = kRounds;
};

const SchedConfig& sched_config()
{
    static const SchedConfig cfg = [] {
        SchedConfig c;  // AIG_SCHED="tail_iters,budget0,round_budget,rounds" overrides (tuning aid)
        if (const char* e = std::getenv("AIG_SCHED")) {
            int a = c.tail_iters, b = c.budget0, r = c.round_budget, n = c.rounds;
            const int got = std::sscanf(e, "%d,%d,%d,%d", &a, &b, &r, &n);
            if (got >= 1 && a >= 0) c.tail_iters = a;
            if (got >= 2 && b >= 1) c.budget0 = b;
            if (got >= 3 && r >= 1) c.round_budget = r;
            if (got >= 4 && n >= 0 && n <= kRounds) c.rounds = n;
        }
        return c;
    }();
    return cfg;
}

int slot_capacity(long long N) { return (int)(N < kMaxSlots ? (N < 1 ? 1 : N) : kMaxSlots); }

size_t round_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// workspace: 64 uint64 counters | checkpoint buffer 0 | checkpoint buffer 1
constexpr size_t kCounterBytes = 64 * sizeof(unsigned long long);
size_t ckpt_buffer_bytes(int cap) { return round_up((size_t)cap * kCkptBytesPerSlot, 256); }

Ckpt ckpt_at(unsigned char* base, int cap)
{
    Ckpt c;
    c.d = reinterpret_cast<double*>(base);
    c.idx = reinterpret_cast<long long*>(base + (size_t)cap * kCkptDoubles * 8);
    c.i = reinterpret_cast<int*>(base + (size_t)cap * (kCkptDoubles * 8 + 8));
    c.cap = cap;
    return c;
}

template <int TRAP, int RESUME, int BLOCK, int MINB>
int stage_capacity(int* blocks_per_sm, int* sm_count)
{
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return AIG_ERR_CUDA;
    if (cudaDeviceGetAttribute(sm_count, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
        return AIG_ERR_CUDA;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(blocks_per_sm, integrate_kernel<TRAP, RESUME, BLOCK, MINB>,
                                                      BLOCK, 0) != cudaSuccess)
        return AIG_ERR_CUDA;
    if (*blocks_per_sm < 1) return AIG_ERR_CUDA;
    return AIG_OK;
}

constexpr int kRoundMinBlocks = kBlock * kBlocksPerSM / kRoundBlock;  // same register budget as stage 0

template <int TRAP>
int launch_integrate(const KParams& K, const double* y0, long long N, const OutPtrs& O, void* workspace,
                     cudaStream_t st)
{
    const SchedConfig& cfg = sched_config();
    const int cap = slot_capacity(N);
    unsigned long long* counters = static_cast<unsigned long long*>(workspace);
    unsigned char* bufs = static_cast<unsigned char*>(workspace) + kCounterBytes;
    const Ckpt buf[2] = {ckpt_at(bufs, cap), ckpt_at(bufs + ckpt_buffer_bytes(cap), cap)};
    if (cudaMemsetAsync(counters, 0, kCounterBytes, st) != cudaSuccess) return AIG_ERR_CUDA;

    int bps = 0, sms = 0;
    int rc = stage_capacity<TRAP, 0, kBlock, kBlocksPerSM>(&bps, &sms);
    if (rc) return rc;
    // stage 0: counters[0] = queue, counters[8] = slots written to buffer 0
    long long blocks = (long long)bps * sms;
    blocks = std::min(blocks, (N + kBlock - 1) / kBlock);
    blocks = std::min(blocks, (long long)std::max(1, cap / kBlock));  // lanes <= slots
    const bool single = (cfg.rounds == 0);
    Sched S;
    S.queue = counters + 0;
    S.n_in = nullptr;
    S.n_out = counters + 8;
    S.in = buf[1];
    S.out = buf[0];
    S.budget = single ? 0x7fffffff : cfg.budget0;
    S.tail_iters = single ? 0x7fffffff : cfg.tail_iters;
    integrate_kernel<TRAP, 0, kBlock, kBlocksPerSM><<<(unsigned)blocks, kBlock, 0, st>>>(K, y0, N, O, S);
    g_kernel_launches++;
    if (cudaGetLastError() != cudaSuccess) return AIG_ERR_CUDA;
    if (single) return AIG_OK;

    // rounds: at most `lanes0` trajectories can be suspended by stage 0, fewer by every later round
    const long long lanes0 = blocks * kBlock;
    rc = stage_capacity<TRAP, 1, kRoundBlock, kRoundMinBlocks>(&bps, &sms);
    if (rc) return rc;
    long long rblocks = std::min((long long)bps * sms, (std::min(lanes0, N) + kRoundBlock - 1) / kRoundBlock);
    long long budget = cfg.round_budget;
    for (int r = 1; r <= cfg.rounds; ++r) {
        Sched R;
        R.queue = counters + 16 + r;
        R.n_in = counters + 8 + (r - 1);
        R.n_out = counters + 8 + r;
        R.in = buf[(r - 1) & 1];
        R.out = buf[r & 1];
        R.budget = (r == cfg.rounds) ? 0x7fffffff : (int)std::min<long long>(budget, 0x7fffffff);
        R.tail_iters = 0x7fffffff;
        integrate_kernel<TRAP, 1, kRoundBlock, kRoundMinBlocks><<<(unsigned)rblocks, kRoundBlock, 0, st>>>(K, y0, N, O, R);
        g_kernel_launches++;
        if (cudaGetLastError() != cudaSuccess) return AIG_ERR_CUDA;
        budget *= 4;
    }
    return AIG_OK;
}

}  // namespace

extern "C" {

int aig_version(void) { return AIG_VERSION; }

uint64_t aig_kernel_launches(void) { return g_kernel_launches.load(); }

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
    // queue / slot counters + two checkpoint buffers of min(N, 65536) suspended trajectories
    return kCounterBytes + 2 * ckpt_buffer_bytes(slot_capacity(N));
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
    OutPtrs O{out->y_final, out->t_final, out->lifetime, out->angle, out->r_min,
              out->n_acc,   out->n_rej,   out->n_turn,   out->status, out->complex_flag};
    switch (trap_mode(p, t_max)) {
        case TRAP_RF: return launch_integrate<TRAP_RF>(K, y0, N, O, workspace, st);
        case TRAP_RF_BIG: return launch_integrate<TRAP_RF_BIG>(K, y0, N, O, workspace, st);
        case TRAP_STATIC: return launch_integrate<TRAP_STATIC>(K, y0, N, O, workspace, st);
        default: return launch_integrate<TRAP_NONE>(K, y0, N, O, workspace, st);
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
    switch (trap_mode(p, p->t0 + 1.0)) {
        case TRAP_RF_BIG:
        case TRAP_RF: step_once_kernel<TRAP_RF><<<blocks, kBlock, 0, st>>>(K, y, t, h, N, ynew, err); break;
        case TRAP_STATIC: step_once_kernel<TRAP_STATIC><<<blocks, kBlock, 0, st>>>(K, y, t, h, N, ynew, err); break;
        default: step_once_kernel<TRAP_NONE><<<blocks, kBlock, 0, st>>>(K, y, t, h, N, ynew, err); break;
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
    const size_t total = 2 * b_y + 4 * b_d + 4 * b_i + flag_bytes + ws_bytes + 8 * (hist_words + edge_words) + 8192;
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
    if (cudaFuncGetAttributes(&fa, integrate_kernel<TRAP_RF, 0, kBlock, kBlocksPerSM>) != cudaSuccess) return AIG_ERR_CUDA;
    int bps = 0, sms = 0;
    const int rc = stage_capacity<TRAP_RF, 0, kBlock, kBlocksPerSM>(&bps, &sms);
    if (rc) return rc;
    if (sm_count) *sm_count = sms;
    if (blocks_per_sm) *blocks_per_sm = bps;
    if (threads_per_block) *threads_per_block = kBlock;
    if (regs_per_thread) *regs_per_thread = fa.numRegs;
    if (local_bytes_per_thread) *local_bytes_per_thread = (int)fa.localSizeBytes;
    return AIG_OK;
}

}  // extern "C"
