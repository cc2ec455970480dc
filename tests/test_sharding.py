"""N > 1 host logic on CPU: world_size-2 ``gloo`` runs of the sharding + histogram reduction that
``bench.py --gpus N`` uses.  The per-shard compute stands in for the GPU:
it is the oracle (tests may call it), so what is checked here is the plumbing -- shards tile the
seeded stream exactly, per-shard results concatenate to the single-process result bit for bit
(trajectories are independent), and ONE all_reduce(sum) of the bins reproduces the
whole-ensemble histogram.
"""
from __future__ import annotations

import os
import socket
import sys

import numpy as np
import pytest

from paper_2509_12381_b200 import inputs, sharding

N_TOTAL = 203  # odd on purpose: ranks own 102 and 101 trajectories


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _hist_torch(h: dict):
    import torch
    return {k: torch.from_numpy(np.ascontiguousarray(h[k]).view(np.int64).copy()) for k in sharding.HIST_KEYS}


def _worker(rank: int, world: int, port: int, tmp: str, per_rank):
    import torch
    import torch.distributed as dist
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    if root not in sys.path:
        sys.path.insert(0, root)
    from oracle import aig_oracle as orc
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = inputs.config(0).replace(N=N_TOTAL)
        y0, lo, hi = sharding.shard_y0(w, rank, world, per_rank=per_rank)
        o = orc.integrate(orc.make_params(**w.params()), y0, w.t_max, w.rtol, w.atol)
        ae, le = inputs.histogram_edges()
        hist = _hist_torch(orc.histogram(o, ae, le, 64))
        sharding.allreduce_hist(hist)
        t_max = sharding.max_over_ranks(1.0 + rank)
        n_sum = sharding.sum_over_ranks(hi - lo)
        np.savez(os.path.join(tmp, f"rank{rank}.npz"), lo=lo, hi=hi, y0=y0, t_max=t_max, n_sum=n_sum,
                 **{"o_" + k: v for k, v in o.items()}, **{"h_" + k: v.numpy() for k, v in hist.items()})
    finally:
        dist.destroy_process_group()


def _run(world, tmp, per_rank):
    import torch.multiprocessing as mp
    mp.spawn(_worker, args=(world, _free_port(), str(tmp), per_rank), nprocs=world, join=True)
    return [np.load(os.path.join(str(tmp), f"rank{r}.npz")) for r in range(world)]


def test_shard_range_tiles_every_index():
    for N in (0, 1, 7, 256, 65536, 4194304 + 3):
        for world in (1, 2, 3, 8):
            r = [inputs.shard_range(N, k, world) for k in range(world)]
            assert r[0][0] == 0 and r[-1][1] == N
            assert all(r[k][1] == r[k + 1][0] for k in range(world - 1))
            sizes = [hi - lo for lo, hi in r]
            assert max(sizes) - min(sizes) <= 1


def test_shards_equal_slices_of_the_single_process_stream():
    w = inputs.config(3).replace(N=1000)
    full = inputs.generate_y0(w)
    for world in (2, 3):
        parts = [sharding.shard_y0(w, r, world) for r in range(world)]
        assert np.array_equal(np.concatenate([p[0] for p in parts], axis=1), full)
    y, lo, hi = sharding.shard_y0(w, 1, 2, per_rank=300)   # weak scaling: rank 1 owns [300, 600)
    assert (lo, hi) == (300, 600) and np.array_equal(y, full[:, 300:600])


def test_flatten_roundtrip():
    import torch
    hist = {k: torch.arange(n, dtype=torch.int64) + 100 * i
            for i, (k, n) in enumerate(zip(sharding.HIST_KEYS, (182, 122, 64, 4, 4)))}
    back = sharding.unflatten_hist(sharding.flatten_hist(hist), hist)
    assert all(torch.equal(back[k], hist[k]) for k in hist)
    assert sharding.allreduce_hist(hist) is hist  # no process group: identity


@pytest.mark.parametrize("per_rank", [None, 96])
def test_world_size_2_gloo(tmp_path, per_rank):
    """Strong split of N_TOTAL (None) and the bench's weak split (96 per rank)."""
    from oracle import aig_oracle as orc
    world = 2
    ranks = _run(world, tmp_path, per_rank)
    n_all = N_TOTAL if per_rank is None else world * per_rank
    assert int(ranks[0]["lo"]) == 0 and int(ranks[-1]["hi"]) == n_all
    assert int(ranks[0]["hi"]) == int(ranks[1]["lo"])
    # single-process result on the same stream
    w = inputs.config(0).replace(N=n_all)
    y0 = inputs.generate_y0(w, n=n_all)
    assert np.array_equal(np.concatenate([r["y0"] for r in ranks], axis=1), y0)
    o = orc.integrate(orc.make_params(**w.params()), y0, w.t_max, w.rtol, w.atol)
    for k, v in o.items():  # per-trajectory outputs need no exchange: concatenation is the result
        cat = np.concatenate([r["o_" + k] for r in ranks], axis=-1)
        assert np.array_equal(cat, v, equal_nan=True), k
    ae, le = inputs.histogram_edges()
    ref = orc.histogram(o, ae, le, 64)
    for r in ranks:  # every rank holds the whole-ensemble histogram after one all_reduce
        for k in sharding.HIST_KEYS:
            assert np.array_equal(r["h_" + k].view(np.uint64), ref[k]), k
        assert int(r["h_totals"][3]) == n_all
        assert float(r["t_max"]) == float(world) and int(r["n_sum"]) == n_all


def test_launch_ranks_refuses_more_ranks_than_devices():
    # what `python bench.py --gpus 2` does on a node with fewer GPUs: fail loudly, launch nothing
    with pytest.raises(SystemExit) as e:
        sharding.launch_ranks("unused.py", [], 2, 1)
    assert "only 1 CUDA device" in str(e.value)
    with pytest.raises(SystemExit):
        sharding.launch_ranks("unused.py", [], 8, 0)


def test_bench_gpus_2_fails_loudly_without_two_gpus():
    import subprocess
    import torch
    if torch.cuda.device_count() >= 2:
        pytest.skip("needs a node with fewer than two GPUs")
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    r = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--steps", "1", "--warmup", "0"],
                       capture_output=True, text=True, env={k: v for k, v in os.environ.items() if k != "WORLD_SIZE"})
    assert r.returncode != 0 and "--gpus 2" in r.stderr and "n_gpus" not in r.stdout


def test_launch_ranks_gloo(capfd):
    """The spawn path of `bench.py --gpus N` (sharding.launch_ranks -> torch.distributed.run -> one process per
    rank), driven with a CPU rank program over gloo: two ranks, each owns 96 trajectories of the stream."""
    import json
    here = os.path.dirname(os.path.abspath(__file__))
    rc = sharding.launch_ranks(os.path.join(here, "gloo_rank_worker.py"), ["96"], 2, 2)
    assert rc == 0
    out = capfd.readouterr().out
    line = json.loads([l for l in out.splitlines() if l.startswith("{")][-1])
    w = inputs.config(0)
    want = sum(int(abs(sharding.shard_y0(w, r, 2, per_rank=96)[0]).sum() * 1e6) for r in range(2))
    assert line == {"n_gpus": 2, "trajectories": 192, "max_over_ranks": 2.0, "checksum": want}
