"""lanczos_shard_update_noalloc (include/hubbard.h): the vector updates of Algorithm 1 (PAPER.md:116-144, lines 4-7
and 11 with eq. 13) with the reduction scratch in the library's fixed `static __device__` array instead of buffers
allocated on first use - for callers that cannot call cudaMalloc.  Checked against the existing path
(lanczos_shard_update) on two calls in a row, against stale contents of the shared array, and at its size limit.

This file is collected LAST on purpose (pytest -x: a failure here must not hide other tests) and
passes alone in a fresh process as well as after the rest of the suite.
"""
import numpy as np
import pytest
import torch

import paper_1204_3425_b200 as hb
from inputs import ring_bonds

pytestmark = pytest.mark.gpu

# relative tolerance on the reduced scalars: fp64 accumulation on both sides, only the cut into partial sums
# differs (tests/test_gpu_parity.py holds H v in fp64 to the same 1e-12)
TOL_SCALAR = 1e-12


def _model(dtype):
    return hb.hubbard_create(8, 4, 4, ring_bonds(8), 1.0, 4.0, dtype)     # the updates only use the model's dtype and GPU


def _vectors(seed, n, tdt):
    g = torch.Generator(device="cpu").manual_seed(seed)
    return [(torch.rand(n, generator=g, dtype=torch.float64) * 2 - 1).to(tdt).cuda() for _ in range(3)]


def _both(m, mode, inout, other, f, coef):
    """(vector, scalar) of the existing path and of the no-alloc path on copies of the same inputs."""
    out = []
    for fn in (m.lanczos_shard_update, m.lanczos_shard_update_noalloc):
        io = inout.clone()
        res = torch.full((1,), float("nan"), dtype=torch.float64, device="cuda")
        fn(mode, io, other, f, coef, res if mode != 2 else None)
        torch.cuda.synchronize()
        out.append((io, float(res.item())))
    return out


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("n", [1, 1000, hb.NOALLOC_CHUNK, 5 * hb.NOALLOC_CHUNK + 77, 3_000_001])
def test_noalloc_matches_existing_path_two_calls_in_a_row(n, dtype):
    tdt = torch.float64 if dtype == "f64" else torch.float32
    m = _model(dtype)
    fprev, hf, f = _vectors(11 + n % 97, n, tdt)
    # call 1: mode 0 (q = H f - b f_prev over f_prev, a = q . f);  call 2, straight after: mode 1 (w = q - a f, |w|^2)
    (q_ref, a_ref), (q_new, a_new) = _both(m, 0, fprev, hf, f, 0.375)
    assert torch.equal(q_ref, q_new)
    assert abs(a_new - a_ref) <= TOL_SCALAR * max(1.0, abs(a_ref))
    (w_ref, s_ref), (w_new, s_new) = _both(m, 1, q_ref, None, f, a_ref)
    assert torch.equal(w_ref, w_new)
    assert abs(s_new - s_ref) <= TOL_SCALAR * max(1.0, abs(s_ref))
    # and against the definition in fp64 on the host (the existing path is itself oracle-tested; this keeps the
    # comparison from being vacuous if both paths were wrong the same way)
    wd = w_new.double().cpu().numpy()
    assert abs(s_new - float(np.dot(wd, wd))) <= 1e-12 * max(1.0, s_new)
    # mode 2 (f_next = w / b) uses no scratch; bit-identical
    (f_ref, _), (f_new, _) = _both(m, 2, w_ref, None, None, 1.0 / np.sqrt(s_ref))
    assert torch.equal(f_ref, f_new)


def test_noalloc_repeated_calls_share_the_array_and_allocate_nothing():
    """The array keeps the last call's partial sums: a small call after a large one must not see them, the same call
    twice gives the same bits, two models share the array, and device memory does not move."""
    m, m2 = _model("f64"), _model("f64")
    big = _vectors(5, 40 * hb.NOALLOC_CHUNK + 3, torch.float64)
    small = _vectors(6, 700, torch.float64)
    res = torch.zeros(4, dtype=torch.float64, device="cuda")
    ios = [big[0].clone(), small[0].clone(), small[0].clone(), small[0].clone()]
    m.lanczos_shard_update_noalloc(1, big[0].clone(), None, big[2], 0.5, res[0:1])      # warm-up: module load
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    m.lanczos_shard_update_noalloc(1, ios[0], None, big[2], 0.5, res[0:1])              # 41 partials written
    m.lanczos_shard_update_noalloc(1, ios[1], None, small[2], 0.5, res[1:2])            # 1 partial: the other 40 are stale
    m.lanczos_shard_update_noalloc(1, ios[2], None, small[2], 0.5, res[2:3])
    m2.lanczos_shard_update_noalloc(1, ios[3], None, small[2], 0.5, res[3:4])           # another model, same array
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0
    r = res.cpu().numpy()
    w = (small[0] - 0.5 * small[2]).cpu().numpy()
    assert abs(r[1] - float(np.dot(w, w))) <= 1e-12 * max(1.0, r[1])
    assert r[1] == r[2] == r[3]
    wb = (big[0] - 0.5 * big[2]).cpu().numpy()
    assert abs(r[0] - float(np.dot(wb, wb))) <= 1e-12 * max(1.0, r[0])


def test_noalloc_rejects_sizes_beyond_its_fixed_scratch():
    m = _model("f32")
    x = torch.ones(16, dtype=torch.float32, device="cuda")
    res = torch.zeros(1, dtype=torch.float64, device="cuda")
    for mode in (0, 1, 2):
        with pytest.raises(hb.HubbardError) as ei:
            m.lanczos_shard_update_noalloc(mode, x, x, x, 1.0, res, n=hb.NOALLOC_MAX_N + 1)     # nothing is enqueued
        assert ei.value.code == hb.ERR_TOO_LARGE and "NOALLOC_MAX_N" in str(ei.value)
    torch.cuda.synchronize()
    assert torch.equal(x, torch.ones_like(x)) and float(res.item()) == 0.0


def test_noalloc_at_the_maximum_size():
    """n = HUBBARD_NOALLOC_MAX_N exactly (fp32: 1 GiB per vector): all 8192 partials in use."""
    n = hb.NOALLOC_MAX_N
    m = _model("f32")
    w = torch.full((n,), 0.5, dtype=torch.float32, device="cuda")
    f = torch.full((n,), 0.25, dtype=torch.float32, device="cuda")
    res = torch.zeros(1, dtype=torch.float64, device="cuda")
    m.lanczos_shard_update_noalloc(1, w, None, f, 1.0, res)           # w = 0.5 - 0.25 = 0.25 exactly; |w|^2 = n / 16
    torch.cuda.synchronize()
    assert float(res.item()) == n / 16.0
    assert float(w[0].item()) == 0.25 and float(w[-1].item()) == 0.25
