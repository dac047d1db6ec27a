"""Pins of the CPU oracle against what the paper and the mathematics fix
(no GPU, no CUDA library).  Each test names the pin of DESIGN.md it covers.

The idea: a plausible mistake anywhere in oracle/ — a dropped term, a wrong
sign (wrap, cross-spin, minus of the Hamiltonian), a wrong index order — must
fail at least one of these.
"""
from math import comb

import numpy as np
import pytest

from conftest import read_golden
from inputs import chain_bonds, g_uniform, ladder_bonds, ring_bonds, torus_bonds
from oracle import hubbard_def as hd
from oracle.lanczos_ref import ground_energy, lanczos, tridiagonal_matrix
from oracle.ref import RefModel


# ---------------------------------------------------------------------- P1
def test_P1_paper_table1_and_eq8():
    sec = hd.Sector(4, 2, 3)
    up_list = [int(x, 2) for x in read_golden("paper_up_list.txt")[0].split()]
    assert sec.states_up == up_list
    for line in read_golden("paper_table1.txt"):
        up, dn, iu, idn, J = line.split()
        up, dn = int(up, 2), int(dn, 2)
        assert sec.pos_up[up] == int(iu)
        assert sec.pos_dn[dn] == int(idn)
        assert sec.J_of_bits(up, dn) == int(J)
        assert sec.bits_of_J(int(J)) == (up, dn)
    assert sec.J_of_bits(0b0101, 0b1101) == 6  # eq. (8)
    # tier 1 enumerates the same lists
    ref = RefModel(4, 2, 3, ring_bonds(4), 1.0, 0.0)
    assert list(ref.states[0]) == sec.states_up and list(ref.states[1]) == sec.states_dn


# ---------------------------------------------------------------------- P2
@pytest.mark.parametrize("t", [1.0, 0.75])
def test_P2_paper_matrix_elements(t):
    H = hd.dense_hamiltonian(4, 2, 3, ring_bonds(4), t, 0.0)
    for line in read_golden("paper_matrix_elements.txt"):
        jp, j, kind, val = line.split()
        got = H[int(jp), int(j)]
        if kind == "abs":
            assert abs(got) == float(val) * t
        else:
            assert got == float(val) * t
    # the state reached from |2> by the up electron hopping 1 -> 2 is |6>
    assert H[2, 6] == -t


# ---------------------------------------------------------------------- P3
def test_P3_dimension_formula():
    for line in read_golden("paper_dims.txt"):
        ns, nu, nd, val, tol = line.split()
        d = comb(int(ns), int(nu)) * comb(int(ns), int(nd))
        assert abs(d - float(val)) <= float(tol) * float(val)
    for ns, nu, nd in [(4, 2, 3), (5, 2, 3), (6, 3, 3), (6, 0, 6), (3, 0, 0)]:
        sec = hd.Sector(ns, nu, nd)
        assert sec.dim == comb(ns, nu) * comb(ns, nd)
        assert sorted(sec.states_up) == sec.states_up
    ref = RefModel(12, 6, 6, ring_bonds(12), 1.0, 4.0)
    assert ref.dim == 853776


# ---------------------------------------------------------------------- P4
SMALL = [
    (4, 2, 3, ring_bonds(4)), (5, 2, 3, ring_bonds(5)), (6, 3, 3, ring_bonds(6)), (6, 2, 3, ladder_bonds(3, 2)),
    (6, 3, 2, ladder_bonds(2, 3) + [(0, 5)]), (4, 2, 2, chain_bonds(4)), (3, 1, 2, ring_bonds(3)),
]


@pytest.mark.parametrize("ns,nu,nd,bonds", SMALL)
def test_P4_hermiticity_exact(ns, nu, nd, bonds):
    H = hd.dense_hamiltonian(ns, nu, nd, bonds, 1.0, 3.0)
    assert np.array_equal(H, H.T)
    # entries are exact sums of +-t and U*k
    assert set(np.unique(H[~np.eye(len(H), dtype=bool)])) <= {-2.0, -1.0, 0.0, 1.0, 2.0}
    assert set(np.unique(np.diag(H))) <= {3.0 * k for k in range(ns + 1)}


# ---------------------------------------------------------------------- P5
@pytest.mark.parametrize("U", [0.0, 4.0, 8.0, -2.5])
def test_P5_two_site_closed_form(U):
    t = 1.0
    H = hd.dense_hamiltonian(2, 1, 1, [(0, 1)], t, U)
    e0 = np.linalg.eigvalsh(H)[0]
    assert abs(e0 - (U - np.sqrt(U * U + 16 * t * t)) / 2) < 1e-13
    if U == 4.0:
        assert abs(e0 - (-0.8284271247)) < 1e-9
    if U == 8.0:
        assert abs(e0 - (-0.4721359550)) < 1e-9


# ---------------------------------------------------------------------- P6
def free_fermion_e0(hopping_levels, n_up, n_dn):
    lv = np.sort(np.asarray(hopping_levels))
    return lv[:n_up].sum() + lv[:n_dn].sum()


def ring_levels(n, t=1.0):
    return [-2 * t * np.cos(2 * np.pi * k / n) for k in range(n)]


def torus_levels(lx, ly, t=1.0):
    return [-2 * t * (np.cos(2 * np.pi * kx / lx) + np.cos(2 * np.pi * ky / ly)) for kx in range(lx) for ky in range(ly)]


@pytest.mark.parametrize("ns,nu,nd", [(4, 2, 3), (5, 2, 3), (6, 3, 3), (6, 2, 4), (6, 1, 1)])
def test_P6_free_fermions_dense_ring(ns, nu, nd):
    """U = 0 on a ring: E0 = sum of the lowest -2t cos k levels per spin.  A wrong
    sign on the periodic wrap (hard-core bosons instead of fermions) changes
    this value for even N_sigma."""
    H = hd.dense_hamiltonian(ns, nu, nd, ring_bonds(ns), 1.0, 0.0)
    assert abs(np.linalg.eigvalsh(H)[0] - free_fermion_e0(ring_levels(ns), nu, nd)) < 1e-12


def test_P6_free_fermions_general_graph():
    """U = 0 on a non-ring bond list: levels of the one-particle hopping matrix."""
    bonds = ladder_bonds(3, 2) + [(0, 5)]
    h1 = np.zeros((6, 6))
    for i, j in bonds:
        h1[i, j] -= 1.0
        h1[j, i] -= 1.0
    H = hd.dense_hamiltonian(6, 3, 2, bonds, 1.0, 0.0)
    assert abs(np.linalg.eigvalsh(H)[0] - free_fermion_e0(np.linalg.eigvalsh(h1), 3, 2)) < 1e-12


def test_P6_free_fermions_tier1_full_scale_C1_C2_C3():
    """Tier 1 at the benchmark sizes, U = 0, against the closed form
    (values also listed in BASELINE.md section 3)."""
    cases = [
        (8, 4, 4, ring_bonds(8), free_fermion_e0(ring_levels(8), 4, 4), -9.656854249492, 80),
        (12, 6, 6, ring_bonds(12), free_fermion_e0(ring_levels(12), 6, 6), -14.928203230276, 160),
        (16, 5, 5, torus_bonds(4, 4), free_fermion_e0(torus_levels(4, 4), 5, 5), -24.0, 90),
    ]
    for ns, nu, nd, bonds, exact, printed, m in cases:
        assert abs(exact - printed) < 1e-9
        ref = RefModel(ns, nu, nd, bonds, 1.0, 0.0)
        v0 = g_uniform(99, np.arange(ref.dim))
        a, b = ref.lanczos_two_vector(v0, m)
        assert abs(ground_energy(a, b) - exact) < 1e-8, (ns, ground_energy(a, b), exact)


# ---------------------------------------------------------------------- P7
@pytest.mark.parametrize("ns,nu,nd", [(4, 3, 3), (4, 2, 2), (5, 4, 3), (4, 2, 3)])
def test_P7_atomic_limit(ns, nu, nd):
    U = 3.0
    H = hd.dense_hamiltonian(ns, nu, nd, ring_bonds(ns), 0.0, U)
    assert np.array_equal(H, np.diag(np.diag(H)))
    assert np.linalg.eigvalsh(H)[0] == U * max(0, nu + nd - ns)
    sec = hd.Sector(ns, nu, nd)
    for J in range(sec.dim):
        u, d = sec.bits_of_J(J)
        assert H[J, J] == U * bin(u & d).count("1")


# ---------------------------------------------------------------------- P8
def jordan_wigner_hamiltonian(ns, bonds, t, U):
    """Independent construction: fermion operators as 2^(2 ns) (sparse) matrices
    (Jordan-Wigner), mode order = the operator order of eq. (4): up sites
    0..ns-1, then down sites 0..ns-1.  Textbook; shares nothing with oracle/."""
    import scipy.sparse as sp

    n_modes = 2 * ns
    I2, Z = sp.identity(2, format="csr"), sp.csr_matrix(np.diag([1.0, -1.0]))
    lower = sp.csr_matrix(np.array([[0.0, 1.0], [0.0, 0.0]]))  # |0><1| : annihilates
    c = []
    for m in range(n_modes):
        mats = [Z] * m + [lower] + [I2] * (n_modes - m - 1)
        op = mats[0]
        for x in mats[1:]:
            op = sp.kron(op, x, format="csr")
        c.append(op)
    H = sp.csr_matrix((2 ** n_modes,) * 2)
    for i, j in bonds:
        for off in (0, ns):
            H = H - t * (c[i + off].T @ c[j + off] + c[j + off].T @ c[i + off])
    for i in range(ns):
        H = H + U * (c[i].T @ c[i]) @ (c[i + ns].T @ c[i + ns])
    return H.tocsr(), c


def fock_vector(c, modes, n_modes):
    """c+_{m0} c+_{m1} ... |O> with the modes in the given left-to-right order."""
    v = np.zeros(2 ** n_modes)
    v[0] = 1.0  # all modes empty = index 0 (basis |0> per mode first)
    for m in reversed(modes):
        v = c[m].T @ v
    return v


@pytest.mark.parametrize("ns,nu,nd,bonds", [
    (4, 2, 3, ring_bonds(4)), (4, 2, 2, ring_bonds(4)), (5, 2, 3, ring_bonds(5)), (5, 3, 1, ring_bonds(5)),
    (6, 3, 3, ring_bonds(6)), (6, 2, 3, ladder_bonds(3, 2)), (6, 3, 2, ladder_bonds(2, 3) + [(0, 5)]),
    (4, 1, 2, [(0, 2), (1, 3), (0, 3)]),
])
def test_P8_dense_brute_force_vs_jordan_wigner(ns, nu, nd, bonds):
    t, U = 1.0, 2.5
    Hfull, c = jordan_wigner_hamiltonian(ns, bonds, t, U)
    sec = hd.Sector(ns, nu, nd)
    B = np.zeros((Hfull.shape[0], sec.dim))
    for J in range(sec.dim):
        u, d = sec.bits_of_J(J)
        modes = [k for k in range(ns) if (u >> k) & 1] + [ns + k for k in range(ns) if (d >> k) & 1]
        B[:, J] = fock_vector(c, modes, 2 * ns)
    Hsec = B.T @ (Hfull @ B)
    assert np.array_equal(B.T @ B, np.eye(sec.dim))
    H = hd.dense_hamiltonian(ns, nu, nd, bonds, t, U)
    assert np.array_equal(H, Hsec)


# ------------------------------------------------- reading Q3: no cross-spin sign
def test_Q3_hop_tables_independent_of_other_spin():
    ns, nu, nd, bonds = 5, 2, 3, ring_bonds(5)
    sec = hd.Sector(ns, nu, nd)
    base_up = hd.hop_table(ns, nu, nd, hd.UP, bonds, 1.0)
    base_dn = hd.hop_table(ns, nu, nd, hd.DN, bonds, 1.0)
    for other in sec.states_dn:
        assert hd.hop_table(ns, nu, nd, hd.UP, bonds, 1.0, other_bits=other) == base_up
    for other in sec.states_up:
        assert hd.hop_table(ns, nu, nd, hd.DN, bonds, 1.0, other_bits=other) == base_dn


def test_eq14_kronecker_sum():
    """PAPER.md:200-206 (eq. 14): H_hop = H_up (x) I + I (x) H_dn, with the
    per-spin tables of the definition."""
    ns, nu, nd, bonds = 5, 2, 3, ring_bonds(5)
    sec = hd.Sector(ns, nu, nd)

    def dense(rows, n):
        M = np.zeros((n, n))
        for r, row in enumerate(rows):
            for cc, v in row:
                M[r, cc] = v
        return M

    Hu = dense(hd.hop_table(ns, nu, nd, hd.UP, bonds, 1.0), sec.dim_up)
    Hd = dense(hd.hop_table(ns, nu, nd, hd.DN, bonds, 1.0), sec.dim_dn)
    H = hd.dense_hamiltonian(ns, nu, nd, bonds, 1.0, 0.0)
    assert np.array_equal(H, np.kron(Hu, np.eye(sec.dim_dn)) + np.kron(np.eye(sec.dim_up), Hd))


# ------------------------------------------------- tier 1 == tier 0 on small sectors
TIER_CASES = SMALL + [(8, 4, 4, ring_bonds(8)), (8, 3, 5, torus_bonds(4, 2)), (6, 3, 3, ring_bonds(6) + [(0, 3)]),
                      (2, 1, 1, [(0, 1)]), (2, 1, 1, [(0, 1), (1, 0)]), (4, 0, 2, ring_bonds(4)), (4, 4, 2, ring_bonds(4))]


@pytest.mark.parametrize("ns,nu,nd,bonds", TIER_CASES)
def test_tier1_tables_bit_exact_vs_tier0(ns, nu, nd, bonds):
    t = 1.0
    ref = RefModel(ns, nu, nd, bonds, t, 0.0)
    for spin in (hd.UP, hd.DN):
        assert ref.hop_rows(spin) == hd.hop_table(ns, nu, nd, spin, bonds, t)


@pytest.mark.parametrize("ns,nu,nd,bonds", TIER_CASES)
def test_tier1_apply_vs_tier0_dense(ns, nu, nd, bonds):
    t, U = 1.0, 4.0
    ref = RefModel(ns, nu, nd, bonds, t, U)
    H = hd.dense_hamiltonian(ns, nu, nd, bonds, t, U)
    x = g_uniform(5, np.arange(ref.dim))
    y = ref.apply(x)
    yd = H @ x
    assert np.abs(y - yd).max() <= 1e-14 * max(1.0, np.abs(yd).max())
    # sampled rows from the definition give the same numbers
    sec = hd.Sector(ns, nu, nd)
    Js = np.unique(np.linspace(0, sec.dim - 1, 7).astype(int))
    ys = hd.sampled_Hv(sec, bonds, t, U, Js, lambda idx: g_uniform(5, idx))
    assert np.abs(ys - yd[Js]).max() <= 1e-14 * max(1.0, np.abs(yd).max())


def test_duplicate_bond_adds():
    """DESIGN.md reading Q6: a bond listed twice adds (effective 2t)."""
    H2 = hd.dense_hamiltonian(2, 1, 1, [(0, 1), (1, 0)], 1.0, 4.0)
    H1 = hd.dense_hamiltonian(2, 1, 1, [(0, 1)], 2.0, 4.0)
    assert np.array_equal(H1, H2)


# ------------------------------------------------- Lanczos oracle
def test_lanczos_krylov_identities():
    """Algorithm 1: with the basis kept, F^T H F = T_m and F^T F = I (short run,
    before orthogonality degrades); lambda_min(T_dim) = lambda_min(H)."""
    H = hd.dense_hamiltonian(6, 2, 2, ring_bonds(6), 1.0, 4.0)
    n = len(H)
    f1 = g_uniform(11, np.arange(n))
    a, b, F = lanczos(lambda x: H @ x, f1, 12, keep_basis=True)
    F = F[:12]
    assert np.abs(F @ F.T - np.eye(12)).max() < 1e-12
    T = tridiagonal_matrix(a, b, 12)
    assert np.abs(F @ H @ F.T - T).max() < 1e-12
    # first coefficients by hand: a_1 = f1^T H f1, b_2 = ||H f1 - a_1 f1||
    f = f1 / np.linalg.norm(f1)
    assert abs(a[0] - f @ H @ f) < 1e-13
    assert abs(b[0] - np.linalg.norm(H @ f - a[0] * f)) < 1e-13
    a, b = lanczos(lambda x: H @ x, f1, 120)
    assert abs(ground_energy(a, b) - np.linalg.eigvalsh(H)[0]) < 1e-11


def test_lanczos_two_vector_variant_matches_algorithm1():
    """eq. 13 (two vectors) is Algorithm 1 re-associated: same a_j, b_j on a
    prefix (reading Q12), same E0."""
    ref = RefModel(8, 4, 4, ring_bonds(8), 1.0, 4.0)
    v0 = g_uniform(12043426, np.arange(ref.dim))
    a3, b3 = lanczos(ref.apply, v0, 100)
    a2, b2 = ref.lanczos_two_vector(v0, 100)
    assert np.abs(a3[:40] - a2[:40]).max() < 1e-10
    assert np.abs(b3[:40] - b2[:40]).max() < 1e-10
    assert abs(ground_energy(a3, b3) - ground_energy(a2, b2)) < 1e-11


def test_lanczos_breakdown_rule():
    """t = 0: H is diagonal with few distinct values; the Krylov space is
    exhausted after that many steps (reading Q11)."""
    ref = RefModel(4, 2, 2, ring_bonds(4), 0.0, 3.0)
    distinct = len(np.unique(ref.apply(np.ones(ref.dim))))
    v0 = g_uniform(3, np.arange(ref.dim))
    a, b = lanczos(ref.apply, v0, 50)
    assert len(a) == distinct
    a2, b2 = ref.lanczos_two_vector(v0, 50)
    assert len(a2) == distinct
    assert abs(ground_energy(a, b) - 0.0) < 1e-9


# ------------------------------------------------- P11 / P9(iv) energies
def test_P11_C1_energy_dense():
    H = hd.dense_hamiltonian(8, 4, 4, ring_bonds(8), 1.0, 4.0)
    e0 = np.linalg.eigvalsh(H)[0]
    assert abs(e0 - (-4.603526299989)) < 2e-11      # SURVEY.md P11 (survey scratch value)
    ref = RefModel(8, 4, 4, ring_bonds(8), 1.0, 4.0)
    a, b = lanczos(ref.apply, g_uniform(12043426, np.arange(ref.dim)), 100)
    assert abs(ground_energy(a, b) - e0) < 1e-10


@pytest.mark.parametrize("U,e_ref", [(4.0, -6.920353562419), (8.0, -3.962563033143)])
def test_P11_C2_energy(U, e_ref):
    ref = RefModel(12, 6, 6, ring_bonds(12), 1.0, U)
    a, b = ref.lanczos_two_vector(g_uniform(12043427, np.arange(ref.dim)), 200)
    assert abs(ground_energy(a, b) - e_ref) < 5e-11


def test_P9_shiba_particle_hole():
    """Bipartite lattice: E0(U; Nup, Ndn) = U*Nup + E0(-U; Nup, Ns-Ndn)."""
    for (nu, nd) in [(3, 3), (2, 3)]:
        U = 4.0
        e1 = np.linalg.eigvalsh(hd.dense_hamiltonian(6, nu, nd, ring_bonds(6), 1.0, U))[0]
        e2 = np.linalg.eigvalsh(hd.dense_hamiltonian(6, nu, 6 - nd, ring_bonds(6), 1.0, -U))[0]
        assert abs(e1 - (U * nu + e2)) < 1e-12


def test_P9_spin_swap_tier1():
    """N_up = N_dn, one bond list: H (V^T) = (H V)^T."""
    ref = RefModel(8, 3, 3, torus_bonds(4, 2), 1.0, 4.0)
    V = g_uniform(8, np.arange(ref.dim)).reshape(ref.dim_up, ref.dim_dn)
    y1 = ref.apply(V.T.copy().ravel()).reshape(ref.dim_up, ref.dim_dn)
    y2 = ref.apply(V.ravel()).reshape(ref.dim_up, ref.dim_dn).T
    assert np.abs(y1 - y2).max() < 1e-13


def test_fig1_ell_worked_example_pins_hop_ell(golden):
    """PAPER.md:208-226 (Fig. 1): the 4x4 example matrix, its ELL `data` / `indices` arrays (width = max nnz per
    row, zero padding printed as *) and their column-major flattening.  Pins RefModel.hop_ell - the CSR -> ELL
    reformatting whose output is the expected value of the library's hubbard_get_hops in tests/test_abi_cpu.py -
    against values the paper prints: a dropped entry, a wrong width, row/column-major confusion or a shifted
    padding would each change the flattened arrays."""
    lines = golden("paper_ell_example.txt")
    k = lines.index("A")
    A = np.array([[float(x) for x in lines[k + 1 + r].split()] for r in range(4)])
    data = lines[lines.index("data_colmajor") + 1].split()
    idx = lines[lines.index("indices_colmajor") + 1].split()
    # the example matrix in CSR, rows in order, columns ascending (as Fig. 1 lists them)
    rp, cj, cv = [0], [], []
    for r in range(4):
        for c in range(4):
            if A[r, c] != 0.0:
                cj.append(c)
                cv.append(A[r, c])
        rp.append(len(cj))
    m = RefModel.__new__(RefModel)                       # hop_ell needs only .csr
    m.csr = {0: (np.array(rp, dtype=np.int64), np.array(cj, dtype=np.int32), np.array(cv, dtype=np.float64))}
    width, cols, vals = m.hop_ell(0)
    assert width == 3 == len(data) // 4                  # "the maximum number of nonzeros per row"
    got_data = vals.T.reshape(-1)                        # column-major flattening
    got_idx = cols.T.reshape(-1)
    for g_d, g_i, w_d, w_i in zip(got_data, got_idx, data, idx):
        if w_d == "*":
            assert g_d == 0.0 and g_i == -1              # padding: the paper zero-fills, the canonical form marks col = -1
        else:
            assert g_d == float(w_d) and g_i == int(w_i)
