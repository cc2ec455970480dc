"""Multi-GPU host logic: one process per GPU, trajectories sharded by index, no data-path collective.

Trajectories never interact; the paper distributes them evenly over workers and
concatenates the results.  Here rank r owns a contiguous index range of the
same seeded stream, integrates it with its own work queue, and the only exchange is ONE
``all_reduce(sum)`` of the few-hundred-bin histogram (KB-sized: latency only, nothing to fuse with).

This module holds no arithmetic of the method and works on CPU tensors with the ``gloo`` backend
(tests/test_sharding.py) exactly as on CUDA tensors with ``nccl`` (bench.py --gpus N).
"""
from __future__ import annotations

import os
import socket
import subprocess
import sys

import numpy as np

from . import inputs

HIST_KEYS = ("angle", "lifetime", "n_turn", "status", "totals")


def shard_y0(w: inputs.Workload, rank: int, world: int, per_rank: int | None = None) -> tuple[np.ndarray, int, int]:
    """Initial conditions of the trajectories rank ``rank`` owns, plus their global range [lo, hi).

    ``per_rank=None``: strong split of the workload's N (``inputs.shard_range``).
    ``per_rank=n``   : weak scaling, rank r owns [r*n, (r+1)*n) of the same stream (bench.py).
    Any shard equals the same columns of a single-process ``generate_y0`` (PCG64.advance).
    """
    if per_rank is None:
        lo, hi = inputs.shard_range(w.N, rank, world)
    else:
        lo, hi = rank * int(per_rank), (rank + 1) * int(per_rank)
    return inputs.generate_y0(w, n=hi - lo, offset=lo), lo, hi


def flatten_hist(hist: dict):
    """Concatenate the histogram arrays in HIST_KEYS order (torch tensors, same device/dtype)."""
    import torch
    return torch.cat([hist[k].reshape(-1) for k in HIST_KEYS])


def unflatten_hist(flat, like: dict) -> dict:
    out, pos = {}, 0
    for k in HIST_KEYS:
        n = like[k].numel()
        out[k] = flat[pos:pos + n].reshape(like[k].shape)
        pos += n
    assert pos == flat.numel()
    return out


def allreduce_hist(hist: dict, group=None) -> dict:
    """Whole-ensemble distribution: one sum over ranks of the concatenated uint64 bins (stored as
    int64 bit patterns; counts stay far below 2^63 so the signed sum is exact).  In place."""
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        return hist
    flat = flatten_hist(hist)
    dist.all_reduce(flat, op=dist.ReduceOp.SUM, group=group)
    for k, v in unflatten_hist(flat, hist).items():
        hist[k].copy_(v)
    return hist


def max_over_ranks(x: float, device="cpu", group=None) -> float:
    """Timing rule of the bench contract: a multi-GPU time is the max over ranks."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        return float(x)
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    return float(t.item())


def sum_over_ranks(x: int, device="cpu", group=None) -> int:
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        return int(x)
    t = torch.tensor([int(x)], dtype=torch.int64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
    return int(t.item())


def free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def launch_ranks(script: str, script_args: list[str], n_ranks: int, n_devices: int, env: dict | None = None) -> int:
    """One process per GPU ("distributed evenly across the ncores cores", one worker per GPU):
    re-launch ``script`` as ``n_ranks`` ranks of one node through ``torch.distributed.run`` (rendezvous on
    127.0.0.1, a free port) and return its exit code.  Fails loudly, without launching anything, when the node has
    fewer devices than ranks: a run must never report fewer GPUs than it was asked for.  Rank r then owns the index
    range ``shard_y0(..., r, n_ranks)`` of the seeded stream; only rank 0 prints."""
    if n_ranks < 1:
        raise SystemExit(f"--gpus {n_ranks}: need at least one rank")
    if n_devices < n_ranks:
        raise SystemExit(f"--gpus {n_ranks}: this node has only {n_devices} CUDA device(s); refusing to run "
                         f"{n_ranks} ranks on fewer GPUs (no rank may share a device)")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n_ranks}",
           "--master-addr", "127.0.0.1", "--master-port", str(free_port()), script, *script_args]
    e = dict(os.environ if env is None else env)
    e.setdefault("NCCL_DEBUG", "INFO")   # one "Init COMPLETE" line per rank on stderr: the ranks can be counted
    e.setdefault("OMP_NUM_THREADS", "1")
    return subprocess.call(cmd, env=e)
