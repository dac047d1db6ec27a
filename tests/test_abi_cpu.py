"""CPU-side checks of libhubbard_b200 (no GPU, no compute calls): the library
loads and exports every symbol include/hubbard.h declares; the host half of
hubbard_create (basis, ranks, hop tables with signs) is bit-exact against the
oracle on all five BASELINE configs and on small irregular sectors; argument
validation; the host tridiagonal eigenvalue routine."""
import ctypes
import re
from pathlib import Path

import numpy as np
import pytest

import paper_1204_3425_b200 as hb
from conftest import read_golden
from inputs import CONFIGS, chain_bonds, ladder_bonds, ring_bonds, torus_bonds
from oracle import hubbard_def as hd
from oracle.ref import RefModel

ROOT = Path(__file__).resolve().parent.parent


def test_every_declared_symbol_is_exported():
    header = (ROOT / "include" / "hubbard.h").read_text()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b((?:hubbard|lanczos)_\w+)\s*\(", header))
    assert declared == set(hb.ABI_SYMBOLS), declared ^ set(hb.ABI_SYMBOLS)
    raw = ctypes.CDLL(hb.LIB_PATH)
    for name in declared:
        assert hasattr(raw, name), name


def test_paper_table1_through_the_abi():
    """PAPER.md:67-95 (Table 1, eq. 8) via hubbard_get_basis."""
    m = hb.hubbard_create_host(4, 2, 3, ring_bonds(4), 1.0, 0.0)
    up, dn = m.hubbard_get_basis(0), m.hubbard_get_basis(1)
    assert list(up) == [int(x, 2) for x in read_golden("paper_up_list.txt")[0].split()]
    for line in read_golden("paper_table1.txt"):
        u, d, iu, idn, J = line.split()
        assert up[int(iu)] == int(u, 2) and dn[int(idn)] == int(d, 2)
        assert int(iu) * m.dim_dn + int(idn) == int(J)
    assert (m.dim_up, m.dim_dn, m.dim) == (6, 4, 24)


def test_paper_matrix_elements_through_the_abi():
    """PAPER.md:77-78,101-102 (eq. 9-10): signs incl. the periodic wrap, from
    the library's own hop tables (H_hop = H_up (x) I + I (x) H_dn, eq. 14)."""
    m = hb.hubbard_create_host(4, 2, 3, ring_bonds(4), 1.0, 0.0)

    def dense(spin, n):
        w, cols, vals = m.hubbard_get_hops(spin)
        M = np.zeros((n, n))
        for r in range(n):
            for k in range(w):
                if cols[r, k] >= 0:
                    M[r, cols[r, k]] = vals[r, k]
        return M

    H = np.kron(dense(0, 6), np.eye(4)) + np.kron(np.eye(6), dense(1, 4))
    for line in read_golden("paper_matrix_elements.txt"):
        jp, j, kind, val = line.split()
        got = H[int(jp), int(j)]
        assert (abs(got) if kind == "abs" else got) == float(val)


@pytest.mark.parametrize("name", ["C1", "C2", "C3", "C4", "C5"])
def test_tables_bit_exact_vs_oracle_on_configs(name):
    c = CONFIGS[name]
    m = hb.hubbard_create_host(c.n_sites, c.n_up, c.n_dn, c.bonds, c.t, c.U_values[0])
    ref = RefModel(c.n_sites, c.n_up, c.n_dn, c.bonds, c.t, c.U_values[0])
    assert (m.dim_up, m.dim_dn, m.dim) == (c.dim_up, c.dim_dn, c.dim)
    for spin in (0, 1):
        assert np.array_equal(m.hubbard_get_basis(spin), ref.states[spin])
        w, cols, vals = m.hubbard_get_hops(spin)
        rw, rc, rv = ref.hop_ell(spin)
        assert w == rw
        assert np.array_equal(cols, rc)
        assert np.array_equal(vals, rv)


IRREGULAR = [
    (4, 2, 3, ring_bonds(4), 1.0), (5, 2, 3, ring_bonds(5), 0.75), (6, 3, 2, ladder_bonds(2, 3) + [(0, 5)], 1.0),
    (2, 1, 1, [(0, 1), (1, 0)], 1.0), (4, 0, 2, ring_bonds(4), 1.0), (4, 4, 2, ring_bonds(4), 1.0),
    (7, 3, 4, ring_bonds(7) + [(0, 3), (6, 2)], 1.3), (8, 3, 5, torus_bonds(4, 2), 1.0), (4, 2, 2, chain_bonds(4), 0.0),
    (1, 1, 0, [], 1.0),
]


@pytest.mark.parametrize("ns,nu,nd,bonds,t", IRREGULAR)
def test_tables_bit_exact_vs_definition_small(ns, nu, nd, bonds, t):
    """Against tier 0 (operator definition), including N_up != N_dn, odd rings,
    a duplicated bond, empty and full sectors, t = 0 and a bond-free site."""
    m = hb.hubbard_create_host(ns, nu, nd, bonds, t, 2.0)
    sec = hd.Sector(ns, nu, nd)
    assert list(m.hubbard_get_basis(0)) == sec.states_up and list(m.hubbard_get_basis(1)) == sec.states_dn
    for spin in (0, 1):
        w, cols, vals = m.hubbard_get_hops(spin)
        rows = hd.hop_table(ns, nu, nd, spin, bonds, t)
        assert w == max((len(r) for r in rows), default=0)
        for r, row in enumerate(rows):
            got = [(int(c), float(v)) for c, v in zip(cols[r], vals[r]) if c >= 0]
            assert got == row
            assert np.all(vals[r][cols[r] < 0] == 0.0)


def test_create_argument_validation():
    bad = [
        dict(n_sites=0, n_up=0, n_dn=0, bonds=[]), dict(n_sites=33, n_up=1, n_dn=1, bonds=[(0, 1)]),
        dict(n_sites=4, n_up=5, n_dn=1, bonds=ring_bonds(4)), dict(n_sites=4, n_up=-1, n_dn=1, bonds=ring_bonds(4)),
        dict(n_sites=4, n_up=2, n_dn=2, bonds=[(0, 4)]), dict(n_sites=4, n_up=2, n_dn=2, bonds=[(1, 1)]),
        dict(n_sites=4, n_up=2, n_dn=2, bonds=[(-1, 2)]),
    ]
    for kw in bad:
        with pytest.raises(hb.HubbardError) as ei:
            hb.hubbard_create_host(t=1.0, U=1.0, **kw)
        assert ei.value.code == -1
    with pytest.raises(hb.HubbardError) as ei:
        hb.hubbard_create_host(4, 2, 2, ring_bonds(4), float("nan"), 1.0)
    assert ei.value.code == -1
    with pytest.raises(hb.HubbardError) as ei:       # C(32,16) = 601080390 fits, C(32,16)... use a sector >= 2^31-1: none at N_s<=32
        hb.hubbard_create_host(4, 2, 2, ring_bonds(4), 1.0, float("inf"))
    assert ei.value.code == -1


def test_host_only_model_refuses_compute():
    m = hb.hubbard_create_host(4, 2, 2, ring_bonds(4), 1.0, 4.0)
    x = np.zeros(m.dim)
    rc = hb.lib.hubbard_apply(m._h, x.ctypes.data, x.ctypes.data, None)
    assert rc == -5
    a = np.zeros(4)
    dp = ctypes.POINTER(ctypes.c_double)
    rc = hb.lib.lanczos_run(m._h, x.ctypes.data, 4, a.ctypes.data_as(dp), a.ctypes.data_as(dp), None, None)
    assert rc == -5
    assert b"no device" in hb.lib.hubbard_strerror(-5)
    m.hubbard_destroy()
    m.hubbard_destroy()  # idempotent
    hb.lib.hubbard_destroy(None)


def test_ground_energy_vs_lapack():
    rng = np.random.default_rng(7)
    for m in (1, 2, 3, 17, 200):
        a = rng.normal(size=m) * 3
        b = np.abs(rng.normal(size=max(m - 1, 1))) + 0.1
        T = np.diag(a) + np.diag(b[:m - 1], 1) + np.diag(b[:m - 1], -1)
        e = hb.lanczos_ground_energy(a, b, m)
        assert abs(e - np.linalg.eigvalsh(T)[0]) <= 1e-13 * max(1.0, np.abs(T).sum(axis=1).max())
    # zero off-diagonals (breakdown leaves beta ~ 0), prefix m < len
    assert hb.lanczos_ground_energy([3.0, -1.0, 2.0], [0.0, 0.0]) == pytest.approx(-1.0, abs=1e-14)
    assert hb.lanczos_ground_energy([3.0, -1.0, 2.0], [0.0, 0.0], 1) == pytest.approx(3.0, abs=1e-14)
    with pytest.raises(hb.HubbardError):
        hb.lanczos_ground_energy([float("nan")], [0.0], 1)


@pytest.mark.parametrize("sorted_", [0, 1, 2])
@pytest.mark.parametrize("lanes,R", [(0, 1), (8, 2), (16, 1), (32, 1), (8, 4)])
@pytest.mark.parametrize("name,ns,nu,nd,bonds", [
    ("C4", 16, 8, 8, torus_bonds(4, 4)), ("C2", 12, 6, 6, ring_bonds(12)), ("odd", 7, 3, 4, ring_bonds(7) + [(0, 3), (2, 6)]),
    ("dup", 6, 3, 3, ring_bonds(6) + [(0, 1)])])
def test_gather_table_is_a_bank_aware_permutation_of_the_hops(name, ns, nu, nd, bonds, lanes, R, sorted_):
    """The device table of variant GATHER (host computation): `perm` is a permutation of the basis states; per
    position the same multiset of (column, sign) as the canonical hop list of its state, columns mapped through
    the inverse permutation (duplicates kept as separate entries); every slot below the warp's exact count holds
    a real entry or a zero slot beyond the tile; counts cover every real entry; and - with scheduling on - the
    lanes of a shared-memory wavefront hit distinct banks up to the reported conflicts."""
    m = hb.hubbard_create_host(ns, nu, nd, bonds, 1.0, 0.0)
    ref = RefModel(ns, nu, nd, bonds, 1.0, 0.0)
    for spin in (0, 1):
        n = m.dim_up if spin == 0 else m.dim_dn
        n_pos = (n + R - 1) // R * R
        g = m.hubbard_get_gather_table(spin, lanes, R, sorted_)
        w, ld, cnt, wsl, perm = g["slots"], g["ld"], g["counts"], g["warp_slots"], g["perm"]
        assert w % 8 == 0 and ld % 32 == 0 and ld >= n_pos and len(wsl) == ld // 32
        assert sorted(perm[:n]) == list(range(n)) and np.all(perm[n:] == -1)
        if not sorted_ or lanes == 0:
            if not sorted_:
                assert np.array_equal(perm[:n], np.arange(n))
        pos = np.empty(n, dtype=np.int64)
        pos[perm[:n]] = np.arange(n)
        flat = g["entries"].transpose(1, 0, 2).reshape(ld, w)            # [position][slot]
        rows = ref.hop_rows(spin)
        n_real = 0
        assert w >= int(wsl.max()) >= 1
        for p in range(ld):
            W = int(wsl[p // 32])
            e = flat[p, :W]
            assert cnt[p] <= W
            real = e[(e >> 1) < n_pos]
            assert np.all((e[(e >> 1) >= n_pos] >> 1) < n_pos + max(lanes, 1))   # zero slots of the tile
            assert np.all((flat[p, cnt[p]:W] >> 1) >= n_pos)                     # beyond the count: padding only
            if p >= n:
                assert len(real) == 0
                continue
            got = {}
            for x in real:                                                      # merge duplicates like the canonical form
                got[int(x >> 1)] = got.get(int(x >> 1), 0.0) + (-1.0 if x & 1 else 1.0)
            want = {int(pos[c]): v for c, v in rows[perm[p]]}
            assert {c: v for c, v in got.items() if v != 0.0} == want
            n_real += len(real)
        if sorted_ == 2 and lanes == 8 and name == "C4":
            # the 4x4 torus has a translation group of 8 elements: almost all states sit in full orbits, the gather
            # costs within 3 % of the ideal sum(hops) / lanes wavefronts and almost nothing collides
            ideal = sum(len(r) for r in rows) / lanes
            assert g["wavefronts"] <= 1.03 * ideal and g["conflicts"] <= n // 10
        if sorted_ == 1 and lanes:
            hops = np.array([sum(1 for _ in rows[perm[p]]) for p in range(n)])
            gmax = [hops[g0:g0 + lanes].max() for g0 in range(0, n - n % lanes, lanes)]
            if name != "dup":                                                    # (merged duplicates change the count)
                assert all(a >= b for a, b in zip(gmax, gmax[1:]))              # groups ordered by their longest row
        if lanes:
            # wavefront groups of `lanes` consecutive positions: distinct banks per slot, up to the reported conflicts
            worst = 0
            for g0 in range(0, ld, lanes):
                W = int(wsl[g0 // 32])
                blk = flat[g0:g0 + lanes, :W] >> 1
                for s in range(W):
                    col = blk[:, s]
                    banks = col[col < n_pos] % lanes
                    worst += len(banks) - len(np.unique(banks))
                    zb = col[col >= n_pos] % lanes                              # a zero slot never shares a bank with a real entry
                    assert not set(zb.tolist()) & set(banks.tolist()) or len(np.unique(banks)) == lanes
            assert worst <= g["conflicts"]
            # the wavefront model: never worse than walking every warp's longest row rounded up to a batch
            per_slot = 32 // lanes
            old_cost = sum(-(-max(int(cnt[w0:w0 + 32].max()), 1) // 8) * 8 * per_slot for w0 in range(0, ld, 32))
            assert g["wavefronts"] <= old_cost


def test_ground_vector_vs_lapack():
    """Host utility: lowest eigenpair of T_m against LAPACK's dense solver, including a
    nearly-degenerate pair and tiny off-diagonals."""
    rng = np.random.default_rng(7)
    cases = [(rng.normal(size=m), np.abs(rng.normal(size=m - 1)) + 0.1) for m in (2, 3, 17, 200)]
    cases.append((np.array([1.0, 1.0 + 1e-9, 3.0]), np.array([1e-7, 0.5])))
    cases.append((np.array([2.0]), np.zeros(0)))
    for a, b in cases:
        e0, y = hb.lanczos_ground_vector(a, b)
        T = np.diag(a) + np.diag(b, 1) + np.diag(b, -1) if len(a) > 1 else np.array([[a[0]]])
        w, v = np.linalg.eigh(T)
        assert abs(e0 - w[0]) <= 1e-12 * max(1.0, np.max(np.abs(w)))
        assert abs(np.linalg.norm(y) - 1.0) < 1e-12 and y[0] >= 0.0
        assert np.max(np.abs(T @ y - e0 * y)) <= 1e-10 * max(1.0, np.max(np.abs(w)))
        if len(a) > 1 and w[1] - w[0] > 1e-6:
            assert abs(abs(np.dot(y, v[:, 0])) - 1.0) < 1e-8


def test_expm_e1_vs_scipy():
    """Host utility of lanczos_propagate: exp(-(tau + i t) T_m) e_1 against scipy's dense matrix exponential."""
    from scipy.linalg import expm
    rng = np.random.default_rng(11)
    for m in (1, 2, 5, 60):
        a = rng.normal(size=m) * 3
        b = np.abs(rng.normal(size=max(m - 1, 0))) + 0.05
        T = np.diag(a) + (np.diag(b, 1) + np.diag(b, -1) if m > 1 else 0)
        for tau, t in ((0.0, 0.7), (0.4, 0.0), (0.2, -1.3)):
            y = hb.lanczos_expm_e1(a, b, tau, t)
            ref = expm(-(tau + 1j * t) * T)[:, 0]
            assert np.max(np.abs(y - ref)) <= 1e-11 * max(1.0, np.max(np.abs(ref)))


def test_debug_knobs_are_explicit_per_model_state(monkeypatch):
    """The test / A-B switches are per-model ABI state (hubbard_debug_set), not environment variables: a stray
    variable cannot reroute a run, unknown keys and out-of-range values are refused."""
    monkeypatch.setenv("HUBBARD_GATHER_R", "1")          # round-1 name: must have no effect any more
    c = CONFIGS["C2"]
    m = hb.hubbard_create_host(c.n_sites, c.n_up, c.n_dn, c.bonds, c.t, 4.0)
    assert m.hubbard_debug_get("gather_R") == 0
    m.hubbard_debug_set("gather_R", 2)
    assert m.hubbard_debug_get("gather_R") == 2
    m2 = hb.hubbard_create_host(c.n_sites, c.n_up, c.n_dn, c.bonds, c.t, 4.0)
    assert m2.hubbard_debug_get("gather_R") == 0         # no process-wide state
    assert m.hubbard_debug_get("gather_fold") == 1       # eight-pass Lanczos form: automatic (where one tile fills the SM)
    m.hubbard_debug_set("gather_fold", 0)
    assert m.hubbard_debug_get("gather_fold") == 0 and m.hubbard_debug_get("resolved_gather_fold") == 0
    for key, bad in (("gather_R", 5), ("gather_ctas", 0), ("no_such_key", 1), ("cluster_NC", -1), ("gather_fold", 3)):
        with pytest.raises(hb.HubbardError):
            m.hubbard_debug_set(key, bad)
    with pytest.raises(hb.HubbardError):
        m.hubbard_debug_get("no_such_key")
    src = "".join(p.read_text() for p in (ROOT / "paper_1204_3425_b200" / "csrc").glob("*"))
    assert "getenv" not in src
