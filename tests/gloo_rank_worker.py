"""Rank program of tests/test_sharding.py::test_launch_ranks_gloo: what bench.py does under
``sharding.launch_ranks``, on CPU with gloo -- ranks from the environment torch.distributed.run sets, each
owns its index range of the seeded stream, one sum over ranks, rank 0 prints one JSON line."""
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import torch.distributed as dist  # noqa: E402

from paper_2509_12381_b200 import inputs, sharding  # noqa: E402

rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo")
per_rank = int(sys.argv[1])
w = inputs.config(0)
y0, lo, hi = sharding.shard_y0(w, rank, world, per_rank=per_rank)
total = sharding.sum_over_ranks(hi - lo)
slowest = sharding.max_over_ranks(float(rank + 1))
checksum = sharding.sum_over_ranks(int(abs(y0).sum() * 1e6))
if rank == 0:
    print(json.dumps({"n_gpus": world, "trajectories": total, "max_over_ranks": slowest, "checksum": checksum}), flush=True)
dist.destroy_process_group()
