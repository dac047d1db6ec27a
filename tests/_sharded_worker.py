"""Worker of tests/test_sharded_cpu.py: the sequencing of the row-sharded Lanczos (paper_1204_3425_b200/sharded.py) on
world_size 2 over gloo, with the vector operations supplied by the ORACLE (numpy + oracle/ref.py: test infrastructure
standing in for the CUDA kernels, which need a GPU).  What is under test is the host logic: the row partition, the
all-gather of unequal shards, the two all-reduces per iteration, the breakdown rule."""
import json
import sys
from pathlib import Path

sys.path.insert(0, str(Path(__file__).resolve().parent.parent))

import numpy as np  # noqa: E402
import torch  # noqa: E402
import torch.distributed as dist  # noqa: E402

from inputs import ring_bonds, start_vector_np  # noqa: E402
from oracle.ref import RefModel  # noqa: E402
from paper_1204_3425_b200 import sharded  # noqa: E402


class OracleOps:
    def __init__(self, ref):
        self.ref = ref

    def empty(self, n):
        return torch.empty(n, dtype=torch.float64)

    def scalar(self):
        return torch.zeros(1, dtype=torch.float64)

    def apply_rows(self, x_full, y_rows, row0, row1):
        y = self.ref.apply(x_full.numpy(), n_threads=1)
        y_rows.copy_(torch.from_numpy(y.reshape(self.ref.dim_up, self.ref.dim_dn)[row0:row1].reshape(-1)))

    def update(self, mode, inout, other, f, coef, result):
        if mode == 0:
            inout.copy_(other - coef * inout)
            result[0] = torch.dot(inout, f)
        elif mode == 1:
            inout.sub_(coef * f)
            result[0] = torch.dot(inout, inout)
        else:
            inout.mul_(coef)


dist.init_process_group(backend="gloo")
rank, world = dist.get_rank(), dist.get_world_size()
ns, nu, nd, t, U, iters = 7, 3, 4, 1.0, 4.0, int(sys.argv[1])        # dim_up = 35: unequal shards on 2 ranks
bonds = ring_bonds(7) + [(0, 3)]
ref = RefModel(ns, nu, nd, bonds, float(sys.argv[2]), U)
v0 = start_vector_np(99, ref.dim)
r0, r1 = sharded.row_partition(ref.dim_up, world)[rank]
shard = torch.from_numpy(v0.reshape(ref.dim_up, ref.dim_dn)[r0:r1].reshape(-1).copy())
alpha, beta = sharded.sharded_lanczos(OracleOps(ref), sharded.TorchDistCollectives(), rank, world, ref.dim_up, ref.dim_dn,
                                      shard, iters)
sys.stdout.write(json.dumps({"rank": rank, "rows": [r0, r1], "alpha": alpha, "beta": beta}) + "\n")
sys.stdout.flush()
dist.destroy_process_group()
