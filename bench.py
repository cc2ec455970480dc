#!/usr/bin/env python
"""bench.py -- throughput of the atom-ion DP5(4) hot path on B200 (BASELINE.json metric).

    python bench.py --gpus N --steps K --warmup W            # our arm (libaig, CUDA)
    python bench.py --impl reference --steps K --warmup W    # the CPU oracle as it stands

One "step" = one pass of the whole hot path (a1-a10) over one batch of
synthetic input: aig_integrate (load, DP5(4) loop, observables, store) + aig_histogram, on
BASELINE.json configs[4] at its central sweep point (N = 4,194,304 trajectories per GPU, config-0
system, q = 0.1, rtol = 1e-10, atol = rtol*1e-2, seed 4).  The other eight points of that
config's 3x3 sweep are run once each after the timed region and reported under "sweep".

Prints ONE JSON line (rank 0).  `value` = trajectories/s over all ranks with inputs resident in
HBM; `e2e` = the same through aig_run_host (pinned HOST buffers in, HOST buffers out, device
allocation + H2D + kernels + D2H inside the timed region); `roofline` = algorithmic FP64
flops of the integrator kernel / its CUDA-event duration against the FP64 non-tensor peak;
`cpu_baseline` = the oracle timed on this box's host cores on a bounded prefix sample.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2509_12381_b200 import inputs  # noqa: E402  (NumPy only)

# SURVEY.md 8(d) / DESIGN.md "Flop accounting": nominal flops of one attempted DP5(4) step of the
# 12-component system as the paper states it (6 f-evals x 38 + 240 stage FMAs + error + controller).
# A LOWER bound on what the kernel executes (ncu counts 996 flops per attempted step, profiles/r02_integrate_full.md):
# the roofline fraction is algorithmic, so the kernel's extra arithmetic earns nothing.
FLOPS_PER_ATTEMPT = 900.0
# 148 SMs x 4 sub-partitions x 16 FP64 FMA lanes x 2 flop x 1.965 GHz (max SM clock)
FP64_PEAK_NOMINAL = 148 * 4 * 16 * 2 * 1.965e9
# dram__bytes_read.sum + dram__bytes_write.sum of one integrate_kernel launch at the bench
# workload, from the ncu --set full capture summarised in profiles/ (None until captured).
INTEGRATE_DRAM_TRAFFIC_BYTES = 8.81e9
INTEGRATE_DRAM_TRAFFIC_SOURCE = ("constant from the ncu --set full capture summarised in profiles/r02_integrate_full.md "
                                 "(the bulk integrator kernel of one call), NOT measured in this run")

WORKLOAD_NAME = "configs[4] N=4194304 q=0.1 rtol=1e-10 atol=1e-12 seed=4"
SWEEP_Q = (0.1, 0.2, 0.4)
SWEEP_RTOL = (1e-8, 1e-10, 1e-12)


def _sig(x, digits=5):
    """Floats to `digits` significant digits, recursively: the driver keeps only the last ~3000 characters of the
    line, and the blocks at its end (sweep, configs, paper_benchmark) must fit there whole."""
    if isinstance(x, float):
        return float(f"{x:.{digits}g}") if np.isfinite(x) else x
    if isinstance(x, dict):
        return {k: _sig(v, digits) for k, v in x.items()}
    if isinstance(x, (list, tuple)):
        return [_sig(v, digits) for v in x]
    if isinstance(x, (np.floating,)):
        return _sig(float(x), digits)
    if isinstance(x, (np.integer,)):
        return int(x)
    return x


def _workload(n, q=0.1, rtol=1e-10):
    w = inputs.config(4, q_trap=q, rtol=rtol)
    return w.replace(N=int(n))


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md)."""

    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")
    NAMES = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")

    def __init__(self, index: int):
        self.rows = []
        self.proc = None
        self.index = index

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.FIELDS}", "--format=csv,noheader,nounits", "-lms", "100",
                 "-i", str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._pump, daemon=True)
        self.thread.start()

    def _pump(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, smax, power, reasons = [], [], [], set()
        for row in self.rows:
            parts = [x.strip() for x in row.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0]))
                smax.append(float(parts[1]))
                power.append(float(parts[2]))
            except ValueError:
                continue
            for name, val in zip(self.NAMES, parts[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None,
                "sm_max_mhz": float(max(smax)) if smax else None,
                "power_w_max": float(max(power)) if power else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def _measured_hbm_gbs():
    """(GB/s, "measured" | "fallback"): HBM copy rate of this pool's B200s as the driver measured it
    (MEASURED_PEAKS.json), else the profiling guide's fallback figure."""
    try:
        with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured"
    except Exception:
        return 6650.0, "fallback"


def _oracle_sample(w, n_sample: int, threads: int):
    """Time the oracle, as it stands, on the first n_sample trajectories of workload w."""
    from oracle import aig_oracle as orc
    y0 = inputs.generate_y0(w, n=n_sample)
    p = orc.make_params(**w.params())
    t0 = time.perf_counter()
    o = orc.integrate(p, y0, w.t_max, w.rtol, w.atol, threads=threads)
    dt = time.perf_counter() - t0
    return dt, int(o["n_acc"].sum()), int(o["n_rej"].sum())


def run_reference(args) -> int:
    """--impl reference: there is no reference implementation to install (the paper's MATLAB sources
    are not in the container); this arm is the CPU oracle, timed as it stands on this box's host cores.
    One step = a bounded prefix sample of the bench workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from oracle import aig_oracle as orc
    orc.build()
    cores = os.cpu_count() or 1
    n_sample = args.ref_sample
    w = _workload(args.n)
    for _ in range(args.warmup):
        _oracle_sample(w, n_sample, cores)
    tot, acc = 0.0, 0
    for _ in range(args.steps):
        dt, a, _r = _oracle_sample(w, n_sample, cores)
        tot += dt
        acc += a
    value = n_sample * args.steps / tot
    sample = f"first {n_sample} trajectories of {WORKLOAD_NAME} per step, {cores} threads (one trajectory per thread at a time)"
    line = {
        "impl": "reference", "metric": "trajectories_per_s", "value": value, "unit": "trajectories/s",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": 1e3 * tot / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": WORKLOAD_NAME, "sample": sample},
        "accepted_steps_per_s": acc / tot,
        "cpu_baseline": {"value": value, "unit": "trajectories/s", "cores": cores, "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": value, "unit": "trajectories/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


def run_ours(args) -> int:
    import torch
    import torch.distributed as dist
    from paper_2509_12381_b200 import binding as aig, sharding

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: CUDA device required (libaig has no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=dev)
    aig.lib()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def max_over_ranks(x: float) -> float:
        return sharding.max_over_ranks(x, dev)

    def sum_over_ranks(x: int) -> int:
        return sharding.sum_over_ranks(x, dev)

    N = int(args.n)                       # trajectories PER GPU (weak scaling)
    w = _workload(N)
    # rank r integrates trajectories [r*N, (r+1)*N) of the same seeded stream (no overlap)
    y0_host = torch.from_numpy(sharding.shard_y0(w, rank, world, per_rank=N)[0]).pin_memory()
    y0 = y0_host.to(dev, non_blocking=True)
    ae, le = inputs.histogram_edges()
    ae_d, le_d = torch.from_numpy(ae).to(dev), torch.from_numpy(le).to(dev)
    out = aig.alloc_out(N, dev)
    ws = torch.zeros(aig.workspace_bytes(N), dtype=torch.uint8, device=dev)
    hist = aig.alloc_hist(len(ae) - 1, len(le) - 1, 64, dev)

    def step(wl, ev=None):
        p = aig.make_params(**wl.params())
        for v in hist.values():
            v.zero_()
        if ev:
            ev[0].record()
        aig.aig_integrate(p, y0, wl.t_max, wl.rtol, wl.atol, out=out, workspace=ws)
        if ev:
            ev[1].record()
        aig.aig_histogram(out, ae_d, le_d, 64, hist=hist)
        if world > 1:  # whole-ensemble distribution: one KB-sized sum over ranks (PAPER.md:485 concatenates on the host)
            sharding.allreduce_hist(hist)

    launches0 = aig.kernel_launches()
    for _ in range(max(args.warmup, 0)):
        step(w)
    barrier()
    launches_warm = aig.kernel_launches()

    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.25)
    kev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    e_begin, e_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e_begin.record()
    for k in range(args.steps):
        step(w, kev[k])
    e_end.record()
    barrier()
    clocks = sampler.stop() if rank == 0 else None
    launches_timed = aig.kernel_launches() - launches_warm
    ms_total = max_over_ranks(e_begin.elapsed_time(e_end))
    ms_each = [a.elapsed_time(b) for a, b in kev]
    ms_int = max_over_ranks(float(np.mean(ms_each)))
    ms_stats = {"min": float(np.min(ms_each)), "median": float(np.median(ms_each)), "max": float(np.max(ms_each)),
                "spread_pct": 100.0 * float(np.max(ms_each) - np.min(ms_each)) / float(np.median(ms_each))}

    def schedule_record(wsp=None):
        """Stage timeline and hand-over counts of the last aig_integrate call (the %globaltimer stamps and
        counters its kernels leave in the workspace): [start, end] in ms of the bulk pass (per-thread
        integrator), the six-lane pass that streams beside it, and the final six-lane pass."""
        cnt = (ws if wsp is None else wsp)[:512].view(torch.int64).cpu().numpy()
        tl = cnt[32:40].astype(np.float64)
        t_first = min((x for x in tl if x > 0), default=0.0)
        st = {name: [round((tl[2 * i] - t_first) / 1e6, 3), round((tl[2 * i + 1] - t_first) / 1e6, 3)]
              for i, name in enumerate(("plan", "bulk", "six_lane_streaming", "six_lane_final")) if tl[2 * i] > 0}
        return st, {"n_handed_over": int(cnt[4]), "taken_by_streaming_pass": int(cnt[61]), "taken_by_final_pass": int(cnt[62]),
                    "class_counts": [int(x) for x in cnt[24:27]]}

    stages_ms, handover = schedule_record()

    def six_lane_step_us(wl, i):
        """Latency of one attempted step of the six-lane integrator: trajectory i of workload wl alone on the
        GPU, handed over at its first step (the schedule hook never changes a result)."""
        y1 = y0[:, i:i + 1].contiguous()
        aig.set_schedule(plan=0, budget=1, tail_iters=0, mean_factor=0, drain_lanes=32)
        try:
            p1 = aig.make_params(**wl.params())
            best = None
            for _ in range(2):
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record()
                o1 = aig.aig_integrate(p1, y1, wl.t_max, wl.rtol, wl.atol)
                b.record()
                torch.cuda.synchronize()
                n1 = int(o1["n_acc"][0].item()) + int(o1["n_rej"][0].item())
                us = a.elapsed_time(b) * 1e3 / max(n1, 1)
                best = us if best is None else min(best, us)
            return best, n1
        finally:
            aig.set_schedule()

    def complex_fraction_r_turn(wl, r_turn):
        """the complex-formation probability when only radial minima inside r_turn count as
        bounces (the graded configs count every radial minimum; far-field micromotion wiggles then count too)."""
        pr = aig.make_params(**{**wl.params(), "r_turn": r_turn})
        aig.aig_integrate(pr, y0, wl.t_max, wl.rtol, wl.atol, out=out, workspace=ws)
        return sum_over_ranks(int(out["complex_flag"].sum(dtype=torch.int64).item())) / (world * N)

    n_acc = int(out["n_acc"].sum(dtype=torch.int64).item())
    n_rej = int(out["n_rej"].sum(dtype=torch.int64).item())
    totals = aig.hist_to_numpy(hist)["totals"] if world == 1 else None
    if totals is not None:
        assert int(totals[0]) == n_acc and int(totals[1]) == n_rej and int(totals[3]) == N
    acc_all, rej_all = sum_over_ranks(n_acc), sum_over_ranks(n_rej)
    n_complex = sum_over_ranks(int(out["complex_flag"].sum(dtype=torch.int64).item()))
    n_tmax = sum_over_ranks(int((out["status"] == 1).sum().item()))
    max_steps_seen = int(max_over_ranks(float(out["n_acc"].max().item())))

    if args.probe_six_lane:
        # only the single-trajectory latency probe (the command of the six-lane kernel's ncu capture in profiles/)
        aig.aig_integrate(aig.make_params(**w.params()), y0, w.t_max, w.rtol, w.atol, out=out, workspace=ws)
        i_probe = int(torch.argmax(out["n_acc"] + out["n_rej"]).item())
        us, n1 = six_lane_step_us(w, i_probe)
        print(json.dumps({"probe": "six_lane_step", "trajectory": i_probe, "attempted_steps": n1, "us_per_step": us,
                          "cycles_per_step_at_1965MHz": us * 1965.0}), flush=True)
        return 0
    i_longest = int(torch.argmax(out["n_acc"] + out["n_rej"]).item())
    max_attempted = int((out["n_acc"][i_longest] + out["n_rej"][i_longest]).item())
    step_us, _ = six_lane_step_us(w, i_longest)
    c50_main = complex_fraction_r_turn(w, 50.0)

    sec = ms_total * 1e-3
    value = world * N * args.steps / sec
    # roofline of the dominant kernel (integrate_kernel), per launch, this rank's launches
    flops_launch = FLOPS_PER_ATTEMPT * (n_acc + n_rej)
    achieved = flops_launch / (ms_int * 1e-3) / 1e12
    peak_meas, _ = aig.fp64_peak_probe(20000, 8)
    info = aig.kernel_info()

    # ---- end to end: HOST buffers through aig_run_host (alloc + H2D + kernels + D2H inside)
    e2e = None
    if not args.no_e2e:
        host_out = {
            "y_final": torch.empty((12, N), dtype=torch.float64).pin_memory(),
            **{k: torch.empty(N, dtype=torch.float64).pin_memory() for k in ("t_final", "lifetime", "angle", "r_min")},
            **{k: torch.empty(N, dtype=torch.int32).pin_memory() for k in ("n_acc", "n_rej", "n_turn", "status")},
            "complex_flag": torch.empty(N, dtype=torch.uint8).pin_memory()}
        host_np = {k: v.numpy() for k, v in host_out.items()}
        p = aig.make_params(**w.params())
        y0_np = y0_host.numpy()
        ne = max(1, min(args.steps, args.e2e_steps))
        aig.aig_run_host(p, y0_np, w.t_max, w.rtol, w.atol, ae, le, 64, out=host_np)  # warm-up
        barrier()
        t0 = time.perf_counter()
        for _ in range(ne):
            res = aig.aig_run_host(p, y0_np, w.t_max, w.rtol, w.atol, ae, le, 64, out=host_np)
        torch.cuda.synchronize()
        dt = max_over_ranks(time.perf_counter() - t0)
        assert int(res["hist"]["totals"][0]) == n_acc  # same kernels, same inputs
        hist_bytes = 8 * sum(len(v) for v in res["hist"].values())
        e2e = {"value": world * N * ne / dt, "unit": "trajectories/s",
               "h2d_bytes_per_step": int(y0_np.nbytes + ae.nbytes + le.nbytes),
               "d2h_bytes_per_step": int(sum(v.nbytes for v in host_np.values() if isinstance(v, np.ndarray)) + hist_bytes),
               "steps": ne, "ms_per_step": 1e3 * dt / ne, "host_memory": "pinned",
               "api": "aig_run_host (C ABI, host pointers)"}
        # where the difference to the device-resident step goes: the two copies timed alone (same pinned buffers, CUDA
        # events), the kernels alone (the timed region above); the rest is cudaMalloc / cudaFree of the ~2 GB slab,
        # the launches and the final synchronisation.  aig_run_host runs them one after the other on one stream.
        def _alone(fn):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            a.record()
            fn()
            b.record()
            torch.cuda.synchronize()
            return a.elapsed_time(b)
        y0_tmp = torch.empty_like(y0)
        h2d_ms = min(_alone(lambda: y0_tmp.copy_(y0_host, non_blocking=True)) for _ in range(2))
        d2h_ms = min(_alone(lambda: [host_out[k].copy_(out[k], non_blocking=True) for k in host_out]) for _ in range(2))
        del y0_tmp
        e2e["breakdown_ms"] = {"h2d_alone": h2d_ms, "kernels_alone": ms_total / args.steps, "d2h_alone": d2h_ms,
                               "rest_malloc_free_launch_sync": e2e["ms_per_step"] - h2d_ms - d2h_ms - ms_total / args.steps}
        del host_out, host_np

    # ---- all nine points of configs[4]'s 3x3 sweep, once each, outside the timed region.  Reported as parallel
    #      arrays (one entry per point, q-major) so that the whole block fits the end of the line.
    #      tail_floor_ms: no call can end before its longest trajectory has taken its steps one after the other =
    #      attempted steps of that trajectory x the latency of one six-lane step (measured above on the bench
    #      workload's longest trajectory, alone on the GPU).  sched_ratio = ms / max(end of the bulk pass, tail floor):
    #      how far the call is from the larger of its two lower bounds under this schedule.
    sweep = None
    if not args.no_sweep:
        cols = ("q", "rtol", "ms", "traj_per_s", "acc_steps_per_s", "frac_fp64_peak", "complex_frac", "complex_frac_r50",
                "max_steps", "tail_floor_ms", "bulk_end_ms", "streaming_end_ms", "final_end_ms", "sched_ratio",
                "handed_over", "taken_by_final_pass")
        sweep = {k: [] for k in cols}
        for q in SWEEP_Q:
            for rtol in SWEEP_RTOL:
                wl = _workload(N, q, rtol)
                ev = (torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
                barrier()
                step(wl, ev)
                barrier()
                ms = max_over_ranks(ev[0].elapsed_time(ev[1]))
                a = sum_over_ranks(int(out["n_acc"].sum(dtype=torch.int64).item()))
                r = sum_over_ranks(int(out["n_rej"].sum(dtype=torch.int64).item()))
                c = sum_over_ranks(int(out["complex_flag"].sum(dtype=torch.int64).item()))
                longest = int(max_over_ranks(float((out["n_acc"] + out["n_rej"]).max().item())))
                tf = FLOPS_PER_ATTEMPT * (a + r) / world / (ms * 1e-3) / 1e12
                st, ho = schedule_record()
                c50 = complex_fraction_r_turn(wl, 50.0)
                floor = longest * step_us * 1e-3
                bulk_end = st.get("bulk", [0.0, 0.0])[1]
                row = (q, rtol, ms, world * N / (ms * 1e-3), a / (ms * 1e-3), tf * 1e12 / FP64_PEAK_NOMINAL,
                       c / (world * N), c50, longest, floor, bulk_end, st.get("six_lane_streaming", [0.0, 0.0])[1],
                       st.get("six_lane_final", [0.0, 0.0])[1], ms / max(bulk_end, floor, 1e-9),
                       ho["n_handed_over"], ho["taken_by_final_pass"])
                for k, v in zip(cols, row):
                    sweep[k].append(v)

    # ---- the other BASELINE.json configs and the paper's own benchmark, outside the timed region (one GPU):
    #      configs[3] (N = 1,048,576, 174/7 amu, q = 0.3, t_max = 1e12: long-lived complexes, step-count imbalance) is
    #      the second throughput config (hard part 2): three calls; configs[0..2] once each (256 and
    #      65,536 trajectories: latency-bound by size); the paper's 2,500-trajectory octant grid.
    configs_rec, paper_rec = None, None
    if world == 1 and not args.no_configs:
        def run_cfg(wl, calls):
            yc = torch.from_numpy(inputs.generate_y0(wl)).to(dev)
            oc = aig.alloc_out(wl.N, dev)
            wc = torch.zeros(aig.workspace_bytes(wl.N), dtype=torch.uint8, device=dev)
            pc = aig.make_params(**wl.params())
            aig.aig_integrate(pc, yc, wl.t_max, wl.rtol, wl.atol, out=oc, workspace=wc)      # warm-up
            torch.cuda.synchronize()
            ts = []
            for _ in range(calls):
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record()
                aig.aig_integrate(pc, yc, wl.t_max, wl.rtol, wl.atol, out=oc, workspace=wc)
                b.record()
                torch.cuda.synchronize()
                ts.append(a.elapsed_time(b))
            ms = float(np.median(ts))
            na = int(oc["n_acc"].sum(dtype=torch.int64).item())
            nr = int(oc["n_rej"].sum(dtype=torch.int64).item())
            longest = int((oc["n_acc"] + oc["n_rej"]).max().item())
            st, ho = schedule_record(wc)
            floor = longest * step_us * 1e-3
            bulk_end = st.get("bulk", [0.0, 0.0])[1]
            return {"N": wl.N, "calls": calls, "ms": ms, "ms_min": float(np.min(ts)), "ms_max": float(np.max(ts)),
                    "traj_per_s": wl.N / (ms * 1e-3), "acc_steps_per_s": na / (ms * 1e-3),
                    "frac_fp64_peak": FLOPS_PER_ATTEMPT * (na + nr) / (ms * 1e-3) / FP64_PEAK_NOMINAL,
                    "mean_steps": na / wl.N, "max_steps": longest, "tail_floor_ms": floor, "bulk_end_ms": bulk_end,
                    "sched_ratio": ms / max(bulk_end, floor, 1e-9),
                    "complex_frac": float(oc["complex_flag"].sum(dtype=torch.int64).item()) / wl.N,
                    "tmax_frac": float((oc["status"] == 1).sum().item()) / wl.N,
                    "handed_over": ho["n_handed_over"], "taken_by_final_pass": ho["taken_by_final_pass"]}
        configs_rec = {"cfg3": run_cfg(inputs.config(3), 3)}
        for i in (0, 1, 2):
            rec = run_cfg(inputs.config(i), 1)
            configs_rec[f"cfg{i}"] = {k: rec[k] for k in ("N", "ms", "traj_per_s", "acc_steps_per_s", "frac_fp64_peak",
                                                          "max_steps", "tail_floor_ms")}
            configs_rec[f"cfg{i}"]["note"] = "latency-bound by size"
        wp = inputs.paper_workload()
        rec = run_cfg(wp, 1)
        paper_rec = {"workload": "50 x 50 octant grid, head-on, tmax 1 ms, rtol 1e-10 (PAPER.md:102, :116)", "N": wp.N,
                     "seconds": rec["ms"] * 1e-3, "acc_steps_per_s": rec["acc_steps_per_s"],
                     "frac_fp64_peak": rec["frac_fp64_peak"], "mean_steps": rec["mean_steps"],
                     "max_steps": rec["max_steps"], "tail_floor_s": rec["tail_floor_ms"] * 1e-3,
                     "complex_frac": rec["complex_frac"]}

    # ---- the widening kernels, outside the timed region: aig_observables and
    #      aig_outliers over the bench workload's results, each timed alone with CUDA events, L2 flushed
    side = None
    if world == 1 and not args.no_side:
        hbm, hbm_kind = _measured_hbm_gbs()
        outp = aig.alloc_out(N, dev, position=True)
        p = aig.make_params(**w.params())
        aig.aig_integrate(p, y0, w.t_max, w.rtol, w.atol, out=outp, workspace=ws)
        extra = aig.aig_observables(p, y0, outp)
        aig.aig_outliers(outp, extra)
        torch.cuda.synchronize()
        flush = torch.empty(2 << 30, dtype=torch.uint8, device=dev)  # also long enough to hide the host side of the next launch
        side = {}
        # algorithmic bytes per trajectory: observables 12 + 3 + 3 doubles in, 4 out; outliers 6 doubles + 2 int32 in
        hist_side = aig.alloc_hist(len(ae) - 1, len(le) - 1, 64, dev)
        map_ue = torch.linspace(0.0, 1.0 + 1e-12, 65, dtype=torch.float64, device=dev)        # 64 x 128 equal-solid-angle cells
        map_pe = torch.linspace(0.0, 2.0 * np.pi, 129, dtype=torch.float64, device=dev)
        map_c = torch.zeros((64, 128), dtype=torch.int64, device=dev)
        map_t = torch.zeros((64, 128), dtype=torch.float64, device=dev)
        # histogram (hot-path row a10): angle, lifetime, four int32 and the flag = 33 B per trajectory
        for name, fn, bpt in (("histogram_kernel", lambda: aig.aig_histogram(outp, ae_d, le_d, 64, hist=hist_side), 33),
                              ("observables_kernel", lambda: aig.aig_observables(p, y0, outp, extra=extra), 176),
                              ("outliers_kernel", lambda: aig.aig_outliers(outp, extra), 56),
                              # map2d: the atom's position (3 doubles) and the value in; the cells stay in L2
                              ("map2d_kernel", lambda: aig.aig_map2d(y0, outp["angle"], map_ue, map_pe, count=map_c, total=map_t), 32)):
            ts = []
            for _ in range(5):
                flush.zero_()
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record()
                fn()
                b.record()
                torch.cuda.synchronize()
                ts.append(a.elapsed_time(b))
            ms = float(np.median(ts))
            gbs = bpt * N / (ms * 1e-3) / 1e9
            side[name] = {"us": round(ms * 1e3, 1), "bytes_per_trajectory": round(bpt, 2), "achieved_gbs": round(gbs, 1),
                          "peak_gbs": hbm, "peak_kind": hbm_kind, "frac": round(gbs / hbm, 3), "bound": "hbm"}
        del outp, extra, flush

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        from oracle import aig_oracle as orc
        orc.build()
        cores = os.cpu_count() or 1
        dt, a, _r = _oracle_sample(w, args.cpu_sample, cores)
        cpu = {"value": args.cpu_sample / dt, "unit": "trajectories/s", "cores": cores, "kind": "oracle",
               "sample": f"first {args.cpu_sample} trajectories of the bench workload, {cores} threads, {dt:.2f} s wall",
               "accepted_steps_per_s": a / dt}
        # the same oracle single-threaded on one core, over a shorter prefix
        n1 = min(args.cpu_sample, 32768)
        dt1, a1, _r1 = _oracle_sample(w, n1, 1)
        cpu["one_core"] = {"value": n1 / dt1, "unit": "trajectories/s", "accepted_steps_per_s": a1 / dt1,
                           "sample": f"first {n1} trajectories, 1 thread, {dt1:.2f} s wall"}

    if rank == 0:
        line = {
            "metric": "trajectories_per_s", "value": value, "unit": "trajectories/s", "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_total / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": WORKLOAD_NAME, "trajectories_per_gpu": N,
                       "l2": "inputs 12*8*N = %d MB and outputs %d MB per step exceed the 126 MB L2; no flush needed"
                             % (96 * N // 2**20, 145 * N // 2**20),
                       "parallelism": f"dp{world} (independent trajectories, contiguous index ranges)"},
            "accepted_steps_per_s": acc_all * args.steps / sec,
            "attempted_steps_per_s": (acc_all + rej_all) * args.steps / sec,
            "mean_accepted_steps": acc_all / (world * N), "max_accepted_steps": max_steps_seen,
            "complex_fraction": n_complex / (world * N), "complex_fraction_r_turn_50": c50_main,
            "tmax_fraction": n_tmax / (world * N),
            "max_attempted_steps": max_attempted, "six_lane_step_us": step_us,
            "tail_floor_ms": max_attempted * step_us * 1e-3, "schedule": handover,
            "ms_integrate_kernel": ms_int,
            "roofline": {"bound": "alu", "achieved": achieved, "peak": FP64_PEAK_NOMINAL / 1e12, "unit": "TFLOP/s",
                         "frac": achieved * 1e12 / FP64_PEAK_NOMINAL, "traffic": INTEGRATE_DRAM_TRAFFIC_BYTES,
                         "traffic_source": INTEGRATE_DRAM_TRAFFIC_SOURCE,
                         "kernel": "aig_integrate: plan kernels + integrate_kernel<TRAP_RF> (bulk) with integrate_split_kernel<TRAP_RF> "
                                   "streaming beside it on a second stream + the final integrate_split_kernel pass, timed as one "
                                   "region on the launching stream",
                         "stages_ms": stages_ms,
                         "flops_per_attempted_step": FLOPS_PER_ATTEMPT,
                         "peak_source": "derived: 148 SM x 64 FP64 FMA lanes x 2 x 1.965 GHz (DESIGN.md)",
                         "peak_measured_dfma": peak_meas / 1e12,
                         "frac_of_measured_dfma": achieved * 1e12 / peak_meas,
                         "hbm_bytes_algorithmic": 241 * N},
            "kernel": info,
            "e2e": e2e, "gpu_launches": int(launches_timed), "clocks": clocks,
            "cpu_baseline": cpu, "side_kernels": side,
            # the blocks the record must show whole come last (the driver keeps the tail of the line)
            "ms_integrate_per_step": ms_stats, "paper_benchmark": paper_rec, "configs": configs_rec, "sweep": sweep,
        }
        print(json.dumps(_sig(line), separators=(",", ":")), flush=True)
    if world > 1:
        dist.destroy_process_group()
    return 0


def main() -> int:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--n", type=int, default=4194304, help="trajectories per GPU (default: configs[4])")
    ap.add_argument("--no-sweep", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-side", action="store_true", help="skip timing aig_observables / aig_outliers")
    ap.add_argument("--no-configs", action="store_true", help="skip configs[0..3] and the paper's own benchmark")
    ap.add_argument("--probe-six-lane", action="store_true",
                    help="run only the latency probe: the workload's longest trajectory alone in the six-lane integrator")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--cpu-sample", type=int, default=2097152)
    ap.add_argument("--ref-sample", type=int, default=262144)
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    world_env = os.environ.get("WORLD_SIZE")
    if world_env is None and args.gpus > 1:
        # python bench.py --gpus N: become N ranks (one process per GPU) of this node
        import torch
        from paper_2509_12381_b200 import sharding
        return sharding.launch_ranks(os.path.abspath(__file__), sys.argv[1:], args.gpus, torch.cuda.device_count())
    if world_env is not None and int(world_env) != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but launched with WORLD_SIZE={world_env}")
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
