"""Row-sharded Lanczos: host-side logic on CPU, world_size 2 over gloo - the path's exchange steps
(all-gather of the row shards, two scalar all-reduces per iteration) with oracle-backed vector operations; the CUDA
kernels behind the same interface are tested on the GPU box (tests/test_gpu_parity.py::test_sharded_*)."""
import numpy as np

from inputs import ring_bonds, start_vector_np
from oracle import lanczos_ref as lr
from oracle.ref import RefModel
from paper_1204_3425_b200 import sharded
from test_bench_dist_cpu import ROOT, _json_lines, _torchrun


def test_row_partition_is_contiguous_and_even():
    for dim_up, world in ((35, 2), (12870, 8), (5, 8), (1, 3)):
        parts = sharded.row_partition(dim_up, world)
        assert len(parts) == world and parts[0][0] == 0 and parts[-1][1] == dim_up
        assert all(a[1] == b[0] for a, b in zip(parts, parts[1:]))
        sizes = [b - a for a, b in parts]
        assert max(sizes) - min(sizes) <= 1


def _oracle(t, iters):
    bonds = ring_bonds(7) + [(0, 3)]
    ref = RefModel(7, 3, 4, bonds, t, 4.0)
    v0 = start_vector_np(99, ref.dim)
    return lr.lanczos(ref.apply, v0, iters)


def test_sharded_lanczos_world2_gloo_matches_algorithm1():
    r = _torchrun([str(ROOT / "tests" / "_sharded_worker.py"), "40", "1.0"])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = _json_lines(r.stdout)
    assert sorted(d["rank"] for d in lines) == [0, 1]
    assert sorted(d["rows"] for d in lines) == [[0, 18], [18, 35]]          # unequal shards
    a_ref, b_ref = _oracle(1.0, 40)
    for d in lines:
        assert len(d["alpha"]) == 40
        assert np.max(np.abs(np.array(d["alpha"][:30]) - a_ref[:30])) <= 1e-10
        assert np.max(np.abs(np.array(d["beta"][:30]) - b_ref[:30])) <= 1e-10
        assert abs(lr.ground_energy(np.array(d["alpha"]), np.array(d["beta"])) - lr.ground_energy(a_ref, b_ref)) <= 1e-10
    assert lines[0]["alpha"] == lines[1]["alpha"] and lines[0]["beta"] == lines[1]["beta"]   # identical on every rank


def test_sharded_lanczos_world2_breakdown():
    """t = 0: the Krylov space is exhausted after a few steps; every rank stops where Algorithm 1 does."""
    r = _torchrun([str(ROOT / "tests" / "_sharded_worker.py"), "50", "0.0"])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = _json_lines(r.stdout)
    a_ref, _ = _oracle(0.0, 50)
    assert len(a_ref) < 50
    for d in lines:
        assert len(d["alpha"]) == len(a_ref)
