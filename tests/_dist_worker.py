"""Worker of tests/test_bench_dist_cpu.py: the host-side multi-rank logic of
bench.py (rank set-up, barrier, max over ranks) on the gloo backend."""
import json
import sys
from pathlib import Path

sys.path.insert(0, str(Path(__file__).resolve().parent.parent))

import torch  # noqa: E402

import bench  # noqa: E402

rank, world, local = bench.dist_setup(2)
bench.barrier(world)
# every rank contributes a different time; all must see the maximum
t = bench.max_over_ranks(10.0 + rank, world, torch.device("cpu"))
# replicas: per-rank work is fixed, the aggregate is world x the per-rank rate at the max time
iters_per_rank = 200
value = world * iters_per_rank / t
sys.stdout.write(json.dumps({"rank": rank, "world": world, "local": local, "t_max": t, "value": value}) + "\n")
sys.stdout.flush()
if world > 1:
    import torch.distributed as dist
    dist.destroy_process_group()
