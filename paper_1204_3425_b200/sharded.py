"""Row-sharded Lanczos over several GPUs (PAPER.md:192 calls multi-GPU "feasible" and names the
obstacle: the H*v needs "a large amount of communication").  One process per GPU, one `hubbard_model` per rank.

V (dim_up x dim_dn, row-major) is split by rows: rank r owns rows [row0_r, row1_r).  Per iteration of Algorithm 1
(eq. 13):

    exchange   f_full  <- all-gather of the shards of f_j                      (the ONE exchange step of the path)
    kernel     y_r      = rows of H f_full                                      hubbard_apply_rows
    kernel     q_r      = y_r - b_j f_{j-1,r}  (over f_{j-1,r}),  a_r = q_r . f_{j,r}      lanczos_shard_update mode 0
    exchange   a_j      = all-reduce(a_r)
    kernel     w_r      = q_r - a_j f_{j,r},   s_r = |w_r|^2                                lanczos_shard_update mode 1
    exchange   b_{j+1}  = sqrt(all-reduce(s_r))
    kernel     f_{j+1,r} = w_r / b_{j+1}                                                    lanczos_shard_update mode 2

This module only sequences those calls and moves the two scalars: every vector operation runs in the library's
kernels (`ops`), every exchange in `torch.distributed` (`coll`).  Both are small interfaces so that the sequencing is
testable without GPUs (tests/test_sharded_cpu.py: world_size 2 over gloo with an oracle-backed `ops`) and the
kernels without a second GPU (tests/test_gpu_parity.py: the ranks' shards processed one after the other on one GPU
with an in-process `coll`).  It has NOT been run on more than one GPU (this build had one): DESIGN.md section 7.
"""
from __future__ import annotations

import math


def row_partition(dim_up: int, world: int):
    """[(row0, row1)] per rank: contiguous, as even as possible."""
    base, extra = divmod(dim_up, world)
    out, r0 = [], 0
    for r in range(world):
        r1 = r0 + base + (1 if r < extra else 0)
        out.append((r0, r1))
        r0 = r1
    return out


class TorchDistCollectives:
    """all-gather / all-reduce over torch.distributed (NCCL between GPUs, gloo in the CPU tests)."""

    def __init__(self, group=None):
        import torch.distributed as dist
        self.dist, self.group = dist, group
        self.rank, self.world = dist.get_rank(group), dist.get_world_size(group)

    def all_gather_rows(self, shard, parts, dim_dn, out_full):
        """out_full[row0_r * dim_dn : row1_r * dim_dn] = rank r's shard, for every r.  Shards may differ in length by
        one row: they travel padded to the longest and are compacted on arrival."""
        import torch
        rows_max = max(r1 - r0 for r0, r1 in parts)
        n_max = rows_max * dim_dn
        send = shard if shard.numel() == n_max else torch.cat([shard, shard.new_zeros(n_max - shard.numel())])
        recv = shard.new_empty(self.world * n_max)
        self.dist.all_gather_into_tensor(recv, send.contiguous(), group=self.group)
        for r, (r0, r1) in enumerate(parts):
            out_full[r0 * dim_dn:r1 * dim_dn].copy_(recv[r * n_max:r * n_max + (r1 - r0) * dim_dn])
        return out_full

    def all_reduce_sum(self, scalar):
        """scalar: 1-element float64 tensor on the compute device; returns the sum over ranks as a Python float."""
        t = scalar.clone()
        self.dist.all_reduce(t, op=self.dist.ReduceOp.SUM, group=self.group)
        return float(t.item())


class LibraryOps:
    """The library's kernels behind the four operations the sequencing needs (argument marshalling only)."""

    def __init__(self, model, device):
        import torch
        self.m, self.torch, self.device = model, torch, device
        self.dtype = torch.float32 if model.dtype_code == 0 else torch.float64

    def empty(self, n):
        return self.torch.empty(n, dtype=self.dtype, device=self.device)

    def scalar(self):
        return self.torch.zeros(1, dtype=self.torch.float64, device=self.device)

    def apply_rows(self, x_full, y_rows, row0, row1):
        self.m.hubbard_apply_rows(x_full, y_rows, row0, row1)

    def update(self, mode, inout, other, f, coef, result):
        self.m.lanczos_shard_update(mode, inout, other, f, coef, result)


def sharded_lanczos(ops, coll, rank, world, dim_up, dim_dn, v0_shard, iters, tau=1e-10):
    """Algorithm 1 on this rank's shard.  v0_shard: this rank's rows of the start vector (need not be normalised; not
    modified).  Returns (alpha, beta) as Python lists - identical on every rank - with the indexing and the breakdown
    rule of lanczos_run (readings Q9, Q11)."""
    parts = row_partition(dim_up, world)
    row0, row1 = parts[rank]
    n = (row1 - row0) * dim_dn
    assert v0_shard.numel() == n
    f, fprev, y = ops.empty(n), ops.empty(n), ops.empty(n)
    f_full = ops.empty(dim_up * dim_dn)
    part = ops.scalar()
    # f_1 = v0 / |v0| (line "Require"), f_0 = 0, b_1 = 0 (lines 1-2)
    f.copy_(v0_shard)
    fprev.zero_()
    ops.update(1, f, None, fprev, 0.0, part)                # w = f - 0 * f_0: leaves |f_r|^2 in `part`
    nrm = math.sqrt(coll.all_reduce_sum(part))
    if not (math.isfinite(nrm) and nrm > 0.0):
        return [], []
    ops.update(2, f, None, None, 1.0 / nrm, None)
    alpha, beta, b, amax = [], [], 0.0, 0.0
    for _ in range(iters):
        coll.all_gather_rows(f, parts, dim_dn, f_full)      # the exchange step
        ops.apply_rows(f_full, y, row0, row1)               # rows of H f_j
        ops.update(0, fprev, y, f, b, part)                 # q over f_{j-1}; a_r
        a = coll.all_reduce_sum(part)
        ops.update(1, fprev, None, f, a, part)              # w over q; |w_r|^2
        bn = math.sqrt(coll.all_reduce_sum(part))
        alpha.append(a)
        beta.append(bn)
        amax = max(amax, abs(a))
        if not math.isfinite(bn) or not (bn > tau * max(1.0, amax)):
            break                                           # lines 8-10
        ops.update(2, fprev, None, None, 1.0 / bn, None)    # line 11
        f, fprev, b = fprev, f, bn
    return alpha, beta
