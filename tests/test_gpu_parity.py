"""GPU parity tests (run on the B200 box with `-m gpu`): the CUDA path, called
through the C ABI (paper_1204_3425_b200.binding -> libhubbard_b200.so), against
the CPU oracle element by element on the same seeded inputs.

Tolerances are BASELINE.json's: H*v relative max-norm error <= 1e-12 (fp64) /
1e-5 (fp32); E_0 after a fixed iteration count <= 1e-10 / 1e-5 relative;
alpha_j, beta_j compared on the prefix of DESIGN.md reading Q12.
"""
import numpy as np
import pytest
import torch

import paper_1204_3425_b200 as hb
from inputs import CONFIGS, chain_bonds, g_uniform, ladder_bonds, ring_bonds, sample_indices, start_vector_torch, torus_bonds
from oracle import hubbard_def as hd
from oracle import lanczos_ref as lr
from oracle.ref import RefModel

pytestmark = pytest.mark.gpu

TOL_HV = {"f64": 1e-12, "f32": 1e-5}
TOL_E0 = {"f64": 1e-10, "f32": 1e-5}
TDT = {"f64": torch.float64, "f32": torch.float32}
VARIANTS = {"paper": hb.VARIANT_PAPER, "twosweep": hb.VARIANT_TWOSWEEP, "gather": hb.VARIANT_GATHER,
            "persist": hb.VARIANT_PERSIST,
            "auto": hb.VARIANT_AUTO}


def oracle_record(name, U):
    """One record of tests/golden/oracle_energies.txt (written by tests/golden/make_energies.py with the oracle
    only): (iterations, E0, alpha prefix, beta prefix)."""
    from conftest import read_golden
    lines = read_golden("oracle_energies.txt")
    for k, line in enumerate(lines):
        f = line.split()
        if f[0] == "case" and f[1] == name and float(f[2]) == float(U):
            assert int(f[4]) == CONFIGS[name].seed
            e0 = float(lines[k + 1].split()[1])
            a = np.array([float(x) for x in lines[k + 2].split()[1:]])
            b = np.array([float(x) for x in lines[k + 3].split()[1:]])
            return int(f[3]), e0, a, b
    raise KeyError((name, U))


def dev():
    assert torch.cuda.is_available(), "these tests need the B200 (no CPU fallback exists)"
    return torch.device("cuda:0")


def start_vector(seed, dim, dtype):
    """Seeded uniform[-1,1) vector, normalised in fp64, rounded to `dtype`
    (reading Q13).  Returns (device tensor, the same bits as fp64 numpy)."""
    v = start_vector_torch(seed, dim, dev(), torch.float64)
    v /= torch.linalg.vector_norm(v)
    v = v.to(TDT[dtype]).contiguous()
    return v, v.double().cpu().numpy()


def rel_max_err(y_gpu, y_ref):
    y = y_gpu.double().cpu().numpy()
    return float(np.max(np.abs(y - y_ref)) / max(np.max(np.abs(y_ref)), 1e-300))


SMALL = [
    (2, 1, 1, [(0, 1)]),
    (4, 2, 3, ring_bonds(4)),
    (5, 2, 3, ring_bonds(5)),
    (6, 3, 3, ring_bonds(6)),
    (6, 2, 4, ladder_bonds(3, 2)),
    (6, 1, 5, chain_bonds(6)),
    (7, 3, 4, ring_bonds(7) + [(0, 3), (2, 6)]),
    (6, 0, 3, ring_bonds(6)),
    (6, 3, 6, ring_bonds(6)),
    (5, 0, 0, ring_bonds(5)),
    (5, 5, 5, ring_bonds(5)),
]


@pytest.mark.parametrize("variant", ["paper", "twosweep", "gather"])
@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("ns,nu,nd,bonds", SMALL)
def test_apply_vs_definition_small(ns, nu, nd, bonds, dtype, variant):
    """H*v against the dense H built from the operator definition (tier 0),
    including N_up != N_dn, odd rings, non-ring bond lists, and the degenerate
    sectors dim_up = 1, dim_dn = 1, dim = 1."""
    t, U = 0.75, 3.5
    H = hd.dense_hamiltonian(ns, nu, nd, bonds, t, U)
    m = hb.hubbard_create(ns, nu, nd, bonds, t, U, dtype)
    m.hubbard_set_variant(VARIANTS[variant])
    assert m.dim == H.shape[0]
    x, x_np = start_vector(77 + ns, m.dim, dtype)
    y = torch.full_like(x, float("nan"))
    m.hubbard_apply(x, y)
    torch.cuda.synchronize()
    y_ref = H @ x_np
    if np.max(np.abs(y_ref)) == 0.0:
        assert float(y.abs().max()) == 0.0
    else:
        assert rel_max_err(y, y_ref) <= TOL_HV[dtype]


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("R", [1, 2])
def test_gather_narrow_tiles(R, dtype):
    """Variant GATHER with tile heights below the 16-byte width (what a large
    sector would get: C5 fp32 has R = 1): H*v on C2 and a short Lanczos run,
    forced through hubbard_debug_set("gather_R")."""
    c = CONFIGS["C2"]
    ref = RefModel(c.n_sites, c.n_up, c.n_dn, c.bonds, c.t, 4.0)
    m = hb.hubbard_create(c.n_sites, c.n_up, c.n_dn, c.bonds, c.t, 4.0, dtype)
    m.hubbard_debug_set("gather_R", R)
    assert m.hubbard_debug_get("resolved_gather_R") == R
    m.hubbard_set_variant(hb.VARIANT_GATHER)
    x, x_np = start_vector(c.seed, c.dim, dtype)
    y = torch.full_like(x, float("nan"))
    m.hubbard_apply(x, y)
    torch.cuda.synchronize()
    assert rel_max_err(y, ref.apply(x_np)) <= TOL_HV[dtype]
    alpha, beta = m.lanczos_run(x, 40)
    a_ref, b_ref = lr.lanczos(ref.apply, x_np, 40)
    assert abs(hb.lanczos_ground_energy(alpha, beta) - lr.ground_energy(a_ref, b_ref)) <= TOL_E0[dtype] * abs(lr.ground_energy(a_ref, b_ref))


@pytest.mark.parametrize("variant", ["paper", "twosweep", "gather"])
@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("name", ["C1", "C2", "C3"])
def test_apply_full_vector_C1_C2_C3(name, dtype, variant):
    c = CONFIGS[name]
    for U in c.U_values:
        ref = RefModel(c.n_sites, c.n_up, c.n_dn, c.bonds, c.t, U)
        m = hb.hubbard_create(c.n_sites, c.n_up, c.n_dn, c.bonds, c.t, U, dtype)
        m.hubbard_set_variant(VARIANTS[variant])
        x, x_np = start_vector(c.seed, c.dim, dtype)
        y = torch.full_like(x, float("nan"))
        m.hubbard_apply(x, y)
        torch.cuda.synchronize()
        assert rel_max_err(y, ref.apply(x_np)) <= TOL_HV[dtype]


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_apply_full_vector_C4(dtype):
    """Headline config at full size, in the launch configuration bench.py
    times (variant AUTO), against the tier-1 oracle over the whole vector."""
    c = CONFIGS["C4"]
    U = 8.0
    ref = RefModel(c.n_sites, c.n_up, c.n_dn, c.bonds, c.t, U)
    m = hb.hubbard_create(c.n_sites, c.n_up, c.n_dn, c.bonds, c.t, U, dtype)
    x, x_np = start_vector(c.seed, c.dim, dtype)
    y = torch.full_like(x, float("nan"))
    m.hubbard_apply(x, y)
    torch.cuda.synchronize()
    y_ref = ref.apply(x_np)
    assert rel_max_err(y, y_ref) <= TOL_HV[dtype]
    # the comparator kernel on the same input
    m.hubbard_set_variant(hb.VARIANT_PAPER)
    y.fill_(float("nan"))
    m.hubbard_apply(x, y)
    torch.cuda.synchronize()
    assert rel_max_err(y, y_ref) <= TOL_HV[dtype]


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_paper_comparator_four_subvectors_per_block(dtype):
    """SURVEY 8(f)-1, second half: the paper's tuned comparator (four sub-vectors per block = four
    elements per thread) - H*v on small ragged sectors (dim_up not a multiple of 4, dim_up < 4) against the dense
    definitional H, on C2 against the tier-1 oracle, and a Lanczos run."""
    for ns, nu, nd, bonds in SMALL:
        H = hd.dense_hamiltonian(ns, nu, nd, bonds, 0.75, 3.5)
        m = hb.hubbard_create(ns, nu, nd, bonds, 0.75, 3.5, dtype)
        m.hubbard_set_variant(hb.VARIANT_PAPER)
        m.hubbard_debug_set("paper_subvectors", 4)
        x, x_np = start_vector(77 + ns, m.dim, dtype)
        y = torch.full_like(x, float("nan"))
        m.hubbard_apply(x, y)
        torch.cuda.synchronize()
        y_ref = H @ x_np
        if np.max(np.abs(y_ref)) == 0.0:
            assert float(y.abs().max()) == 0.0
        else:
            assert rel_max_err(y, y_ref) <= TOL_HV[dtype]
    c = CONFIGS["C2"]
    ref = RefModel(c.n_sites, c.n_up, c.n_dn, c.bonds, c.t, 4.0)
    m = hb.hubbard_create(c.n_sites, c.n_up, c.n_dn, c.bonds, c.t, 4.0, dtype)
    m.hubbard_set_variant(hb.VARIANT_PAPER)
    m.hubbard_debug_set("paper_subvectors", 4)
    x, x_np = start_vector(c.seed, c.dim, dtype)
    y = torch.full_like(x, float("nan"))
    m.hubbard_apply(x, y)
    torch.cuda.synchronize()
    assert rel_max_err(y, ref.apply(x_np)) <= TOL_HV[dtype]
    alpha, beta = m.lanczos_run(x, 60)
    a_ref, b_ref = lr.lanczos(ref.apply, x_np, 60)
    n = 30
    tol_c = 1e-10 if dtype == "f64" else 1e-5
    assert np.max(np.abs(alpha[:n] - a_ref[:n]) / np.maximum(1.0, np.abs(a_ref[:n]))) <= tol_c
    e_ref = lr.ground_energy(a_ref, b_ref)
    assert abs(hb.lanczos_ground_energy(alpha, beta) - e_ref) <= TOL_E0[dtype] * abs(e_ref)


def _sampled_parity(name, dtype, n_samples, U):
    """Pin P10: (H v0)[J] on seeded sample indices from the operator
    definition (tier 0), v0[J] = g(seed, J) un-normalised."""
    c = CONFIGS[name]
    m = hb.hubbard_create(c.n_sites, c.n_up, c.n_dn, c.bonds, c.t, U, dtype)
    x = start_vector_torch(c.seed, c.dim, dev(), TDT[dtype])
    y = torch.empty_like(x)
    m.hubbard_apply(x, y)
    torch.cuda.synchronize()
    J = sample_indices(c.seed + 1000, c.dim, n_samples)
    sec = hd.Sector(c.n_sites, c.n_up, c.n_dn)

    def v_of(idx):
        v = g_uniform(c.seed, idx)
        return v.astype(np.float32).astype(np.float64) if dtype == "f32" else v

    y_ref = hd.sampled_Hv(sec, c.bonds, c.t, U, J, v_of)
    y_s = y[torch.from_numpy(J).to(dev())].double().cpu().numpy()
    scale = float(y.abs().max())
    assert np.max(np.abs(y_s - y_ref)) / scale <= TOL_HV[dtype]
    return m, x, y


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_apply_sampled_vs_definition_C4(dtype):
    _sampled_parity("C4", dtype, 600, 4.0)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_apply_sampled_vs_definition_C5(dtype):
    """dim = 2 363 904 400 > 2^31: 64-bit offsets; V row larger than one SM's
    shared memory in fp64."""
    free, _ = torch.cuda.mem_get_info()
    need = 2 * CONFIGS["C5"].dim * (8 if dtype == "f64" else 4) + (4 << 30)
    if free < need:
        pytest.skip(f"needs {need >> 30} GiB of free HBM")
    _sampled_parity("C5", dtype, 300, 4.0)
    torch.cuda.empty_cache()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_full_scale_invariants_C4(dtype):
    """Pin P9 at full scale, oracle-free: Hermiticity, U-linearity of the
    diagonal with its closed form, spin-swap H(V^T) = (H V)^T."""
    c = CONFIGS["C4"]
    tol = 1e-11 if dtype == "f64" else 2e-5
    m = hb.hubbard_create(c.n_sites, c.n_up, c.n_dn, c.bonds, c.t, 8.0, dtype)
    x, _ = start_vector(c.seed, c.dim, dtype)
    z, _ = start_vector(c.seed + 7, c.dim, dtype)
    hx, hz = torch.empty_like(x), torch.empty_like(x)
    m.hubbard_apply(x, hx)
    m.hubbard_apply(z, hz)
    a = torch.dot(z.double(), hx.double()).item()
    b = torch.dot(hz.double(), x.double()).item()
    scale = torch.linalg.vector_norm(hx.double()).item() * torch.linalg.vector_norm(z.double()).item()
    assert abs(a - b) / scale <= tol
    # (ii) H(U) x - H(0) x = U popcount(up & dn) o x
    m.hubbard_set_U(0.0)
    h0 = torch.empty_like(x)
    m.hubbard_apply(x, h0)
    st_up = torch.from_numpy(m.hubbard_get_basis(0).astype(np.int64)).to(dev())
    st_dn = torch.from_numpy(m.hubbard_get_basis(1).astype(np.int64)).to(dev())
    diff = (hx.double() - h0.double()).view(m.dim_up, m.dim_dn)
    ymax = hx.abs().max().item()
    worst = 0.0
    for r0 in range(0, m.dim_up, 1024):
        r1 = min(m.dim_up, r0 + 1024)
        both = st_up[r0:r1, None] & st_dn[None, :]
        docc = torch.zeros_like(both)
        for k in range(c.n_sites):
            docc += (both >> k) & 1
        want = 8.0 * docc.double() * x.view(m.dim_up, m.dim_dn)[r0:r1].double()
        worst = max(worst, (diff[r0:r1] - want).abs().max().item())
    assert worst / ymax <= tol
    # (iii) spin swap (N_up = N_dn, one bond list)
    m.hubbard_set_U(8.0)
    xt = x.view(m.dim_up, m.dim_dn).t().contiguous().view(-1)
    hxt = torch.empty_like(x)
    m.hubbard_apply(xt, hxt)
    err = (hxt.view(m.dim_dn, m.dim_up).t() - hx.view(m.dim_up, m.dim_dn)).abs().max().item()
    assert err / ymax <= tol


def _lanczos_case(name, U, dtype, variant, iters, n_prefix):
    c = CONFIGS[name]
    ref = RefModel(c.n_sites, c.n_up, c.n_dn, c.bonds, c.t, U)
    m = hb.hubbard_create(c.n_sites, c.n_up, c.n_dn, c.bonds, c.t, U, dtype)
    m.hubbard_set_variant(VARIANTS[variant])
    v0, v0_np = start_vector(c.seed, c.dim, dtype)
    keep = v0.clone()
    alpha, beta = m.lanczos_run(v0, iters)
    assert torch.equal(v0, keep), "lanczos_run must not modify v0"
    a_ref, b_ref = lr.lanczos(ref.apply, v0_np, iters)
    assert len(alpha) == len(a_ref) == iters
    tol_c = 1e-10 if dtype == "f64" else 1e-5
    n = min(n_prefix, iters)
    assert np.max(np.abs(alpha[:n] - a_ref[:n]) / np.maximum(1.0, np.abs(a_ref[:n]))) <= tol_c
    assert np.max(np.abs(beta[:n] - b_ref[:n]) / np.maximum(1.0, np.abs(b_ref[:n]))) <= tol_c
    e_gpu = hb.lanczos_ground_energy(alpha, beta)
    e_ref = lr.ground_energy(a_ref, b_ref)
    assert abs(e_gpu - e_ref) / abs(e_ref) <= TOL_E0[dtype]
    return e_gpu


@pytest.mark.parametrize("variant", ["paper", "twosweep", "gather", "persist", "auto"])
def test_lanczos_C1(variant):
    e = _lanczos_case("C1", 4.0, "f64", variant, 100, 50)
    assert abs(e - (-4.603526299989)) < 1e-9          # SURVEY P11, also dense eigvalsh in the CPU suite


@pytest.mark.parametrize("variant", ["paper", "twosweep", "gather", "persist", "auto"])
@pytest.mark.parametrize("dtype,n_prefix", [("f64", 50), ("f32", 30)])
@pytest.mark.parametrize("U", [4.0, 8.0])
def test_lanczos_C2(U, dtype, n_prefix, variant):
    _lanczos_case("C2", U, dtype, variant, 200, n_prefix)


@pytest.mark.parametrize("dtype,n_prefix", [("f64", 40), ("f32", 30)])
def test_lanczos_persist_on_a_larger_sector(dtype, n_prefix):
    """PERSIST forced on C3 (19 M elements, many elements per thread, several blocks per SM's worth of work)."""
    _lanczos_case("C3", 8.0, dtype, "persist", 40, n_prefix)


@pytest.mark.parametrize("dtype,n_prefix", [("f64", 40), ("f32", 30)])
def test_lanczos_C3_prefix(dtype, n_prefix):
    """C3 with a shortened run (the oracle's H*v costs ~0.3 s here): prefix of
    alpha/beta and E_0^(m) at m = 40."""
    _lanczos_case("C3", 8.0, dtype, "auto", 40, n_prefix)


def _lanczos_vs_golden(name, U, dtype, n_prefix):
    """Full-length run in the launch configuration bench.py times (variant AUTO) against the stored oracle run
    (Algorithm 1 verbatim on the tier-1 H*v, same seeded start vector): E_0 after the configuration's fixed
    iteration count (north_star: <= 1e-10 / 1e-5 relative) and the coefficient prefix of reading Q12."""
    c = CONFIGS[name]
    iters, e_ref, a_ref, b_ref = oracle_record(name, U)
    assert iters == c.iters
    m = hb.hubbard_create(c.n_sites, c.n_up, c.n_dn, c.bonds, c.t, U, dtype)
    v0, _ = start_vector(c.seed, c.dim, dtype)
    alpha, beta = m.lanczos_run(v0, iters)
    assert len(alpha) == iters
    tol_c = 1e-10 if dtype == "f64" else 1e-5
    n = min(n_prefix, len(a_ref))
    assert np.max(np.abs(alpha[:n] - a_ref[:n]) / np.maximum(1.0, np.abs(a_ref[:n]))) <= tol_c
    assert np.max(np.abs(beta[:n] - b_ref[:n]) / np.maximum(1.0, np.abs(b_ref[:n]))) <= tol_c
    e_gpu = hb.lanczos_ground_energy(alpha, beta)
    assert abs(e_gpu - e_ref) <= TOL_E0[dtype] * abs(e_ref)
    return e_gpu


@pytest.mark.parametrize("dtype,n_prefix", [("f64", 50), ("f32", 30)])
def test_lanczos_C3_full_vs_oracle(dtype, n_prefix):
    """C3 at its full 200 iterations."""
    e = _lanczos_vs_golden("C3", 8.0, dtype, n_prefix)
    assert abs(e - (-17.510366694879)) < 1e-4            # SURVEY P11 (sanity only)


@pytest.mark.parametrize("dtype,n_prefix", [("f64", 50), ("f32", 30)])
@pytest.mark.parametrize("U", [4.0, 8.0])
def test_lanczos_C4_full_vs_oracle(U, dtype, n_prefix):
    """The headline configuration: E_0 after the fixed 200 iterations, U = 4 and U = 8, both dtypes."""
    _lanczos_vs_golden("C4", U, dtype, n_prefix)


def _c5_fits(dtype, n_vec):
    free, _ = torch.cuda.mem_get_info()
    need = n_vec * CONFIGS["C5"].dim * (8 if dtype == "f64" else 4) + (4 << 30)
    if free < need:
        pytest.skip(f"needs {need >> 30} GiB of free HBM")


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_lanczos_C5_first_iterations_vs_oracle(dtype):
    """C5 (dim = 2 363 904 400 > 2^31) through lanczos_run under AUTO - the cluster (DSMEM) row sweep in its
    Lanczos form for fp64, the row-major gather ROW sweep for fp32, the <LZ> strip sweep and the axpy+norm kernel
    with 64-bit offsets: a_1, b_2, a_2, b_3 against Algorithm 1 written out on the tier-1 oracle over the FULL
    vector (tests/golden/make_energies.py C5: two resident host vectors of 18.9 GB)."""
    _c5_fits(dtype, 3)
    c = CONFIGS["C5"]
    iters, _, a_ref, b_ref = oracle_record("C5", 4.0)
    m = hb.hubbard_create(c.n_sites, c.n_up, c.n_dn, c.bonds, c.t, 4.0, dtype)
    assert m.hubbard_debug_get("resolved_variant") == hb.VARIANT_TWOSWEEP
    v0 = start_vector_torch(c.seed, c.dim, dev(), TDT[dtype])     # un-normalised: lanczos_run normalises its copy
    alpha, beta = m.lanczos_run(v0, iters)
    del v0
    tol = 1e-10 if dtype == "f64" else 1e-5
    assert len(alpha) == iters == 2
    assert np.max(np.abs(alpha - a_ref) / np.maximum(1.0, np.abs(a_ref))) <= tol
    assert np.max(np.abs(beta - b_ref) / np.maximum(1.0, np.abs(b_ref))) <= tol
    m.close()
    torch.cuda.empty_cache()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_lanczos_C5_free_fermions(dtype):
    """Pin P6 at full scale, oracle-free: U = 0 on the half-filled 18-ring, E_0 = 2 * sum of the 9 lowest levels
    of -2 cos(2 pi n / 18) = -23.035081932575 (closed shell).  Any wrong wrap sign, 32-bit offset or DSMEM
    index would move it."""
    _c5_fits(dtype, 3)
    c = CONFIGS["C5"]
    e_exact = 2.0 * sum(sorted(-2.0 * np.cos(2.0 * np.pi * np.arange(18) / 18.0))[:9])
    assert abs(e_exact - (-23.035081932575)) < 1e-11
    m = hb.hubbard_create(c.n_sites, c.n_up, c.n_dn, c.bonds, c.t, 0.0, dtype)
    v0 = start_vector_torch(c.seed, c.dim, dev(), TDT[dtype])
    alpha, beta, e0 = m.lanczos_run_until(v0, 300, check_every=20, tol=1e-13 if dtype == "f64" else 1e-7)
    del v0
    assert abs(e0 - e_exact) <= TOL_E0[dtype] * abs(e_exact), (len(alpha), e0)
    m.close()
    torch.cuda.empty_cache()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("ctas", [1, 2, 4])
@pytest.mark.parametrize("name,ns,nu,nd,bonds", [("C2", 12, 6, 6, ring_bonds(12)), ("odd", 13, 5, 7, ring_bonds(13) + [(0, 5)])])
def test_gather_lanczos_folded_and_nine_pass_forms(name, ns, nu, nd, bonds, ctas, dtype):
    """Variant GATHER has two Lanczos forms: the folded one (default: the ROW sweep parks its tile of
    u_j in tensor memory and applies line 4's - b_{j+1} f_j itself, with b_{j+1}^2 = |q_j|^2 - a_j^2 from the COL
    sweep before; 8 vector passes) and the nine-pass one (gather_fold = 0: the COL sweep reads u_j).  Both against
    Algorithm 1 of the oracle, with 1, 2 and 4 CTAs per SM sharing the SM's 512 tensor-memory columns."""
    ref = RefModel(ns, nu, nd, bonds, 1.0, 4.0)
    x, x_np = start_vector(78, ref.dim, dtype)
    a_ref, b_ref = lr.lanczos(ref.apply, x_np, 40)
    e_ref = lr.ground_energy(a_ref, b_ref)
    tol_c = 1e-10 if dtype == "f64" else 1e-5
    got = {}
    for fold in (2, 0):
        m = hb.hubbard_create(ns, nu, nd, bonds, 1.0, 4.0, dtype)
        m.hubbard_set_variant(hb.VARIANT_GATHER)
        m.hubbard_debug_set("gather_ctas", ctas)
        assert m.hubbard_debug_get("resolved_gather_fold") == 0 or ctas == 1     # automatic: only one CTA per SM folds
        m.hubbard_debug_set("gather_fold", fold)
        cols = m.hubbard_debug_get("resolved_gather_fold")
        assert (cols >= 32 and cols & (cols - 1) == 0 and cols * ctas <= 512) if fold else cols == 0
        alpha, beta = m.lanczos_run(x, 40)
        n = 30
        assert np.max(np.abs(alpha[:n] - a_ref[:n]) / np.maximum(1.0, np.abs(a_ref[:n]))) <= tol_c
        assert np.max(np.abs(beta[:n] - b_ref[:n]) / np.maximum(1.0, np.abs(b_ref[:n]))) <= tol_c
        assert abs(hb.lanczos_ground_energy(alpha, beta) - e_ref) <= TOL_E0[dtype] * abs(e_ref)
        a2, b2 = m.lanczos_run(x, 40)
        assert np.array_equal(alpha, a2) and np.array_equal(beta, b2)      # deterministic, and tensor memory is released
        got[fold] = (alpha, beta)
        if fold and m.hubbard_debug_get("resolved_gather_fold"):
            # the folded COL sweep with its first entry batches from L2 instead of tensor memory: the same arithmetic
            m.hubbard_debug_set("gather_tmem_entries", 0)
            a3, b3 = m.lanczos_run(x, 40)
            assert np.array_equal(alpha, a3) and np.array_equal(beta, b3)
    # the two forms differ only in rounding (the coefficient of f_j is |q|^2 - a^2 instead of |w|^2)
    assert np.max(np.abs(got[0][0][:30] - got[2][0][:30])) <= tol_c * 20


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("name,ns,nu,nd,bonds", [("C2", 12, 6, 6, ring_bonds(12)), ("odd", 13, 5, 7, ring_bonds(13) + [(0, 5)])])
def test_auto_twosweep_with_gather_row(name, ns, nu, nd, bonds, dtype):
    """The path C5 fp32 takes under AUTO, on sectors the oracle covers in full: the gather tile is narrower than
    16 bytes (forced with gather_R = 1), so AUTO resolves to TWOSWEEP whose row half is the gather ROW sweep in
    its ROW-MAJOR Lanczos form (eq. 13 folded: y = c (t H_dn + D) x - b_j c_{j-1} y), followed by the <LZ> strip
    sweep and the axpy+norm kernel."""
    ref = RefModel(ns, nu, nd, bonds, 1.0, 4.0)
    m = hb.hubbard_create(ns, nu, nd, bonds, 1.0, 4.0, dtype)
    m.hubbard_debug_set("gather_R", 1)
    m.hubbard_debug_set("persist_max_dim", 0)
    assert m.hubbard_debug_get("resolved_gather_R") == 1
    assert m.hubbard_debug_get("resolved_variant") == hb.VARIANT_TWOSWEEP
    x, x_np = start_vector(77, m.dim, dtype)
    y = torch.full_like(x, float("nan"))
    m.hubbard_apply(x, y)
    torch.cuda.synchronize()
    assert rel_max_err(y, ref.apply(x_np)) <= TOL_HV[dtype]
    m.hubbard_profile(True)
    alpha, beta = m.lanczos_run(x, 40)
    kt = m.hubbard_kernel_times()
    m.hubbard_profile(False)
    assert kt["row_sweep"][0] == 40 and kt["col_sweep"][0] == 40 and kt["vec_sweep"][0] == 40
    a_ref, b_ref = lr.lanczos(ref.apply, x_np, 40)
    tol_c = 1e-10 if dtype == "f64" else 1e-5
    n = 30
    assert np.max(np.abs(alpha[:n] - a_ref[:n]) / np.maximum(1.0, np.abs(a_ref[:n]))) <= tol_c
    assert np.max(np.abs(beta[:n] - b_ref[:n]) / np.maximum(1.0, np.abs(b_ref[:n]))) <= tol_c
    e_ref = lr.ground_energy(a_ref, b_ref)
    assert abs(hb.lanczos_ground_energy(alpha, beta) - e_ref) <= TOL_E0[dtype] * abs(e_ref)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_lanczos_C4_free_fermions(dtype):
    """Pin P6 at full scale, oracle-free: U = 0 on the 4x4 half-filled torus,
    E_0 = -24 (two copies of the lowest 8 levels of -2(cos kx + cos ky)).
    Wrong wrap signs would give hard-core-boson energies instead.  The
    single-particle levels are -4, -2, 0, 2, 4, so H has only the 25 distinct
    eigenvalues -24, -22, ..., 24: the Krylov space is exhausted after 25
    steps and lanczos_run must stop there (Algorithm 1 lines 8-10, reading Q11)."""
    c = CONFIGS["C4"]
    m = hb.hubbard_create(c.n_sites, c.n_up, c.n_dn, c.bonds, c.t, 0.0, dtype)
    v0, _ = start_vector(c.seed, c.dim, dtype)
    alpha, beta = m.lanczos_run(v0, 200)
    if dtype == "f64":
        assert len(alpha) == 25
    else:
        assert 25 <= len(alpha) <= 200
    e = hb.lanczos_ground_energy(alpha, beta)
    tol = 1e-10 if dtype == "f64" else 1e-5
    assert abs(e + 24.0) <= 24.0 * tol


def test_lanczos_breakdown_atomic_limit():
    """t = 0: H is diagonal with few distinct values; the Krylov space is
    exhausted and lanczos_run stops early (Algorithm 1 lines 8-10, reading
    Q11) exactly where the oracle does."""
    ns, nu, nd, bonds = 6, 3, 3, ring_bonds(6)
    ref = RefModel(ns, nu, nd, bonds, 0.0, 4.0)
    for variant in ("paper", "twosweep", "gather", "persist"):
        m = hb.hubbard_create(ns, nu, nd, bonds, 0.0, 4.0, "f64")
        m.hubbard_set_variant(VARIANTS[variant])
        v0, v0_np = start_vector(5, m.dim, "f64")
        alpha, beta = m.lanczos_run(v0, 50)
        a_ref, b_ref = lr.lanczos(ref.apply, v0_np, 50)
        assert len(alpha) == len(a_ref) < 50
        assert abs(hb.lanczos_ground_energy(alpha, beta) - 0.0) < 1e-9     # U * max(0, N - N_s) = 0


def test_edge_cases_and_errors():
    m = hb.hubbard_create(6, 3, 3, ring_bonds(6), 1.0, 4.0, "f64")
    x, _ = start_vector(1, m.dim, "f64")
    with pytest.raises(hb.HubbardError):
        m.hubbard_apply(x, x)                               # aliasing
    a, b = m.lanczos_run(x, 0)
    assert len(a) == 0 and len(b) == 0
    # zero start vector: no iteration can be done
    a, b = m.lanczos_run(torch.zeros_like(x), 5)
    assert len(a) == 0
    # host-buffer entry points give the same bits as the device ones
    y = torch.empty_like(x)
    m.hubbard_apply(x, y)
    torch.cuda.synchronize()
    yh = np.empty(m.dim)
    m.hubbard_apply_host(x.cpu().numpy(), yh)
    assert np.array_equal(yh, y.cpu().numpy())
    a1, b1 = m.lanczos_run(x, 20)
    a2, b2 = m.lanczos_run_host(x.cpu().numpy(), 20)
    assert np.array_equal(a1, a2) and np.array_equal(b1, b2)
    # run-to-run determinism of the reductions
    a3, b3 = m.lanczos_run(x, 20)
    assert np.array_equal(a1, a3) and np.array_equal(b1, b3)
    assert m.hubbard_launch_count() > 0


def test_non_default_stream():
    c = CONFIGS["C2"]
    m = hb.hubbard_create(c.n_sites, c.n_up, c.n_dn, c.bonds, c.t, 4.0, "f64")
    x, _ = start_vector(c.seed, c.dim, "f64")
    y0, y1 = torch.empty_like(x), torch.empty_like(x)
    m.hubbard_apply(x, y0)
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        m.hubbard_apply(x, y1)
    s.synchronize()
    torch.cuda.synchronize()
    assert torch.equal(y0, y1)


# ---------------------------------------------------------------- SURVEY 8(f)-2
def _double_occupancy(psi_np, st_up, st_dn):
    docc = np.array([[bin(int(u) & int(d)).count("1") for d in st_dn] for u in st_up], dtype=np.float64)
    return float(np.sum(docc.reshape(-1) * psi_np * psi_np))


@pytest.mark.parametrize("variant", ["paper", "twosweep", "gather", "persist"])
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_ground_state_vector_small(dtype, variant):
    """lanczos_ground_state against the dense eigenvector of the definitional H (tier 0) on a sector with a
    non-degenerate ground state: overlap, energy, residual |H psi - E psi| and the double occupancy
    <sum_i n_iup n_idn> (eq. 2)."""
    ns, nu, nd, bonds, t, U = 6, 3, 3, ring_bonds(6), 1.0, 4.0
    H = hd.dense_hamiltonian(ns, nu, nd, bonds, t, U)
    w, v = np.linalg.eigh(H)
    assert w[1] - w[0] > 1e-3
    m = hb.hubbard_create(ns, nu, nd, bonds, t, U, dtype)
    m.hubbard_set_variant(VARIANTS[variant])
    v0, _ = start_vector(11, m.dim, dtype)
    psi = torch.empty_like(v0)
    # 60 iterations: E_0 has converged, and the accumulated vector is not yet degraded by the loss of
    # orthogonality that follows convergence (the ORACLE's own residual goes 3e-15 at m = 60 -> 1.3e-11 at m = 80,
    # DESIGN.md section 5), so the bound below is a statement about the kernels, not about Lanczos
    e0, done = m.lanczos_ground_state(v0, 60, psi)
    tol = 1e-9 if dtype == "f64" else 2e-4
    assert abs(e0 - w[0]) <= (1e-10 if dtype == "f64" else 1e-5) * abs(w[0])
    p = psi.double().cpu().numpy()
    assert abs(np.linalg.norm(p) - 1.0) < (1e-12 if dtype == "f64" else 1e-6)
    assert abs(abs(np.dot(p, v[:, 0])) - 1.0) <= tol
    assert np.max(np.abs(H @ p - e0 * p)) <= (1e-7 if dtype == "f64" else 1e-3)
    st_up, st_dn = m.hubbard_get_basis(0), m.hubbard_get_basis(1)
    # an observable is linear in the vector error (the overlap is quadratic in it)
    assert abs(_double_occupancy(p, st_up, st_dn) - _double_occupancy(v[:, 0], st_up, st_dn)) <= (1e-6 if dtype == "f64" else 2e-3)


def test_ground_state_vector_C2_vs_oracle_eigsh():
    """C2 (dim 853 776): the ground vector from the CUDA path against the oracle's matrix-free H with a
    library eigensolver (scipy ARPACK on oracle.ref.RefModel.apply)."""
    from scipy.sparse.linalg import LinearOperator, eigsh
    c = CONFIGS["C2"]
    ref = RefModel(c.n_sites, c.n_up, c.n_dn, c.bonds, c.t, 4.0)
    m = hb.hubbard_create(c.n_sites, c.n_up, c.n_dn, c.bonds, c.t, 4.0, "f64")
    v0, v0_np = start_vector(c.seed, c.dim, "f64")
    psi = torch.empty_like(v0)
    e0, done = m.lanczos_ground_state(v0, 200, psi)
    assert done == 200
    w, v = eigsh(LinearOperator((c.dim, c.dim), matvec=ref.apply, dtype=np.float64), k=1, which="SA", v0=v0_np, tol=1e-12)
    assert abs(e0 - w[0]) <= 1e-10 * abs(w[0])
    p = psi.double().cpu().numpy()
    assert abs(abs(np.dot(p, v[:, 0])) - 1.0) <= 1e-8
    # the library's own H on its own vector: Rayleigh quotient = E_0, small residual
    hp = torch.empty_like(psi)
    m.hubbard_apply(psi, hp)
    torch.cuda.synchronize()
    assert abs(torch.dot(psi, hp).item() - e0) <= 1e-10 * abs(e0)
    assert (hp - e0 * psi).abs().max().item() <= 1e-6


@pytest.mark.parametrize("variant", ["twosweep", "gather", "persist"])
def test_run_until_converges_and_matches_fixed_run(variant):
    """Convergence-driven stopping: stops well before the iteration cap, returns the same
    alpha/beta as a fixed run of that length (bit-identical: same kernels, same order) and E_0 within tol."""
    c = CONFIGS["C2"]
    m = hb.hubbard_create(c.n_sites, c.n_up, c.n_dn, c.bonds, c.t, 4.0, "f64")
    m.hubbard_set_variant(VARIANTS[variant])
    v0, _ = start_vector(c.seed, c.dim, "f64")
    a, b, e0 = m.lanczos_run_until(v0, 400, check_every=10, tol=1e-11)
    n = len(a)
    assert 30 <= n < 400 and n % 10 == 0
    a2, b2 = m.lanczos_run(v0, n)
    assert np.array_equal(a, a2) and np.array_equal(b, b2)
    assert abs(e0 - hb.lanczos_ground_energy(a, b)) == 0.0
    assert abs(e0 - (-6.920353562419)) < 1e-8                        # SURVEY P11 / oracle test_P11_C2_energy
    # the cap is honoured and a breakdown ends the run (t = 0)
    a3, b3, _ = m.lanczos_run_until(v0, 25, check_every=10, tol=0.0)
    assert len(a3) == 25
    m0 = hb.hubbard_create(6, 3, 3, ring_bonds(6), 0.0, 4.0, "f64")
    m0.hubbard_set_variant(VARIANTS[variant])
    x, _ = start_vector(5, m0.dim, "f64")
    a4, b4, e4 = m0.lanczos_run_until(x, 50, check_every=3, tol=0.0)
    a5, b5 = m0.lanczos_run(x, 50)
    assert len(a4) == len(a5) < 50 and abs(e4) < 1e-9


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_lanczos_C4_prefix_vs_oracle(dtype):
    """Headline configuration at full size in the launch configuration bench.py times (variant AUTO = the two
    gather sweeps): the first Lanczos coefficients against Algorithm 1 run verbatim on the tier-1 oracle's H*v."""
    c = CONFIGS["C4"]
    n = 6
    ref = RefModel(c.n_sites, c.n_up, c.n_dn, c.bonds, c.t, 8.0)
    m = hb.hubbard_create(c.n_sites, c.n_up, c.n_dn, c.bonds, c.t, 8.0, dtype)
    v0, v0_np = start_vector(c.seed, c.dim, dtype)
    alpha, beta = m.lanczos_run(v0, n)
    a_ref, b_ref = lr.lanczos(ref.apply, v0_np, n)
    tol = 1e-10 if dtype == "f64" else 1e-5
    assert len(alpha) == n
    assert np.max(np.abs(alpha - a_ref) / np.maximum(1.0, np.abs(a_ref))) <= tol
    assert np.max(np.abs(beta - b_ref) / np.maximum(1.0, np.abs(b_ref))) <= tol


# ---------------------------------------------------------------- SURVEY 8(f)-4
@pytest.mark.parametrize("variant", ["paper", "twosweep", "gather", "persist"])
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_propagate_small_vs_dense_exponential(dtype, variant):
    """lanczos_propagate against exp(-(tau + i t) H) v from the dense eigen-decomposition of the
    definitional H (tier 0): real time, imaginary time and both; norm conservation in real time."""
    ns, nu, nd, bonds, tt, U = 6, 3, 3, ring_bonds(6), 1.0, 4.0
    H = hd.dense_hamiltonian(ns, nu, nd, bonds, tt, U)
    w, Q = np.linalg.eigh(H)
    m = hb.hubbard_create(ns, nu, nd, bonds, tt, U, dtype)
    m.hubbard_set_variant(VARIANTS[variant])
    v0, v0_np = start_vector(21, m.dim, dtype)
    v0 *= 1.7                                           # the propagated vector must carry |v0|
    v0_np = v0.double().cpu().numpy()
    tol = 1e-9 if dtype == "f64" else 2e-4
    for tau, t in ((0.0, 0.35), (0.25, 0.0), (0.1, -0.2)):
        ref = Q @ (np.exp(-(tau + 1j * t) * w) * (Q.T @ v0_np))
        re, im = torch.empty_like(v0), torch.empty_like(v0)
        done = m.lanczos_propagate(v0, 60, tau, t, re, im)
        assert done >= 1
        got = re.double().cpu().numpy() + 1j * im.double().cpu().numpy()
        assert np.max(np.abs(got - ref)) <= tol * np.max(np.abs(ref))
        if tau == 0.0:
            assert abs(np.linalg.norm(got) - np.linalg.norm(v0_np)) <= tol * np.linalg.norm(v0_np)
    # imaginary part not requested
    re2 = torch.empty_like(v0)
    m.lanczos_propagate(v0, 60, 0.25, 0.0, re2, None)
    ref = Q @ (np.exp(-0.25 * w) * (Q.T @ v0_np))
    assert np.max(np.abs(re2.double().cpu().numpy() - ref)) <= tol * np.max(np.abs(ref))


@pytest.mark.parametrize("variant", ["paper", "twosweep", "gather", "persist", "auto"])
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_propagate_complex_small_vs_dense_exponential(dtype, variant):
    """lanczos_propagate_complex (a second step of a time propagation: the state is complex) against
    exp(-(tau + i t) H) psi from the dense eigen-decomposition of the definitional H (tier 0), complex psi; a real
    psi (im = None) reproduces lanczos_propagate; in-place continuation; N_up != N_dn."""
    for ns, nu, nd, bonds in ((6, 3, 3, ring_bonds(6)), (6, 2, 4, ladder_bonds(3, 2))):
        tt, U = 1.0, 4.0
        H = hd.dense_hamiltonian(ns, nu, nd, bonds, tt, U)
        w, Q = np.linalg.eigh(H)
        m = hb.hubbard_create(ns, nu, nd, bonds, tt, U, dtype)
        m.hubbard_set_variant(VARIANTS[variant])
        xr, _ = start_vector(31, m.dim, dtype)
        xi, _ = start_vector(32, m.dim, dtype)
        xr *= 1.3
        xi *= 0.6
        psi0 = xr.double().cpu().numpy() + 1j * xi.double().cpu().numpy()
        tol = 1e-9 if dtype == "f64" else 2e-4
        for tau, t in ((0.0, 0.35), (0.2, -0.15)):
            ref = Q @ (np.exp(-(tau + 1j * t) * w) * (Q.T @ psi0))
            re, im = torch.empty_like(xr), torch.empty_like(xr)
            done = m.lanczos_propagate_complex(xr, xi, 60, tau, t, re, im)
            assert done >= 1
            got = re.double().cpu().numpy() + 1j * im.double().cpu().numpy()
            assert np.max(np.abs(got - ref)) <= tol * np.max(np.abs(ref))
            if tau == 0.0:
                assert abs(np.linalg.norm(got) - np.linalg.norm(psi0)) <= tol * np.linalg.norm(psi0)
        # real start vector: the same result as lanczos_propagate
        re1, im1, re2, im2 = (torch.empty_like(xr) for _ in range(4))
        m.lanczos_propagate(xr, 60, 0.0, 0.3, re1, im1)
        m.lanczos_propagate_complex(xr, None, 60, 0.0, 0.3, re2, im2)
        scale = float(xr.abs().max())
        assert float((re1 - re2).abs().max()) <= tol * scale and float((im1 - im2).abs().max()) <= tol * scale
        # two steps in place == one step of the summed time
        a, b = xr.clone(), xi.clone()
        m.lanczos_propagate_complex(a, b, 60, 0.0, 0.2, a, b)
        m.lanczos_propagate_complex(a, b, 60, 0.0, 0.15, a, b)
        ref = Q @ (np.exp(-1j * 0.35 * w) * (Q.T @ psi0))
        got = a.double().cpu().numpy() + 1j * b.double().cpu().numpy()
        assert np.max(np.abs(got - ref)) <= 2 * tol * np.max(np.abs(ref))


def test_propagate_complex_C2_two_steps_vs_oracle_taylor():
    """C2 at full size: two propagation steps (the second from a complex state) against the Taylor series of
    exp(-i (t1 + t2) H) v evaluated with the ORACLE's matrix-free H; unitarity."""
    c = CONFIGS["C2"]
    m = hb.hubbard_create(c.n_sites, c.n_up, c.n_dn, c.bonds, c.t, 4.0, "f64")
    ref = RefModel(c.n_sites, c.n_up, c.n_dn, c.bonds, c.t, 4.0)
    v0, v0_np = start_vector(c.seed, c.dim, "f64")
    re, im = torch.empty_like(v0), torch.empty_like(v0)
    t1, t2 = 0.03, 0.02
    m.lanczos_propagate(v0, 30, 0.0, t1, re, im)
    m.lanczos_propagate_complex(re, im, 30, 0.0, t2, re, im)
    psi = re.double().cpu().numpy() + 1j * im.double().cpu().numpy()
    assert abs(np.linalg.norm(psi) - 1.0) <= 1e-10
    t = t1 + t2
    term, acc = v0_np.astype(complex), v0_np.astype(complex)
    for k in range(1, 31):
        term = (-1j * t / k) * (ref.apply(term.real) + 1j * ref.apply(term.imag))
        acc = acc + term
    assert np.max(np.abs(psi - acc)) <= 1e-10 * np.max(np.abs(acc))


def test_propagate_C2_properties():
    """C2 at full size (no dense exponential): unitarity in real time and agreement with the Taylor series of
    exp(-i t H) v evaluated with the oracle's matrix-free H."""
    c = CONFIGS["C2"]
    m = hb.hubbard_create(c.n_sites, c.n_up, c.n_dn, c.bonds, c.t, 4.0, "f64")
    ref = RefModel(c.n_sites, c.n_up, c.n_dn, c.bonds, c.t, 4.0)
    v0, v0_np = start_vector(c.seed, c.dim, "f64")
    re, im = torch.empty_like(v0), torch.empty_like(v0)
    t = 0.05
    m.lanczos_propagate(v0, 30, 0.0, t, re, im)
    psi = re.double().cpu().numpy() + 1j * im.double().cpu().numpy()
    assert abs(np.linalg.norm(psi) - 1.0) <= 1e-10
    # Taylor series of exp(-i t H) v with the ORACLE's H*v (t |H| ~ 1.5: 30 terms are far past convergence)
    term, acc = v0_np.astype(complex), v0_np.astype(complex)
    for k in range(1, 31):
        term = (-1j * t / k) * (ref.apply(term.real) + 1j * ref.apply(term.imag))
        acc = acc + term
    assert np.max(np.abs(psi - acc)) <= 1e-10 * np.max(np.abs(acc))


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("R,NC", [(0, 0), (1, 2), (1, 4), (2, 2), (2, 4)])
@pytest.mark.parametrize("name,ns,nu,nd,bonds", [("C2", 12, 6, 6, ring_bonds(12)), ("odd", 13, 5, 7, ring_bonds(13) + [(0, 5)])])
def test_cluster_row_sweep(name, ns, nu, nd, bonds, R, NC, dtype):
    """The distributed-shared-memory row sweep (clusters of NC CTAs holding R rows, kernels_cluster.cuh: what
    C5 fp64 uses because a V row exceeds one SM) forced on sectors the oracle covers in full: H*v and a Lanczos
    run; dim_dn not a multiple of 32 or of the cluster split, N_up != N_dn, odd dim_up with R = 2."""
    ref = RefModel(ns, nu, nd, bonds, 1.0, 4.0)
    m = hb.hubbard_create(ns, nu, nd, bonds, 1.0, 4.0, dtype)
    m.hubbard_debug_set("force_cluster_row", 1)
    m.hubbard_debug_set("cluster_R", R)
    m.hubbard_debug_set("cluster_NC", NC)
    assert m.hubbard_debug_get("resolved_cluster_row") == 1 and m.hubbard_debug_get("resolved_gather_R") == 0
    if R:
        assert (m.hubbard_debug_get("resolved_cluster_R"), m.hubbard_debug_get("resolved_cluster_NC")) == (R, NC)
    x, x_np = start_vector(77, m.dim, dtype)
    y = torch.full_like(x, float("nan"))
    m.hubbard_apply(x, y)
    torch.cuda.synchronize()
    assert rel_max_err(y, ref.apply(x_np)) <= TOL_HV[dtype]
    assert m.hubbard_kernel_times is not None
    m.hubbard_profile(True)
    alpha, beta = m.lanczos_run(x, 40)
    assert m.hubbard_kernel_times()["row_sweep"][0] == 40          # the cluster kernel is the row sweep of every iteration
    m.hubbard_profile(False)
    a_ref, b_ref = lr.lanczos(ref.apply, x_np, 40)
    e_ref = lr.ground_energy(a_ref, b_ref)
    assert abs(hb.lanczos_ground_energy(alpha, beta) - e_ref) <= TOL_E0[dtype] * abs(e_ref)


# ---------------------------------------------------------------- SURVEY 8(f)-3
@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("name,ns,nu,nd,bonds", [("C2", 12, 6, 6, ring_bonds(12)), ("odd", 7, 3, 4, ring_bonds(7) + [(0, 3), (2, 6)])])
def test_sharded_apply_rows(name, ns, nu, nd, bonds, dtype):
    """hubbard_apply_rows: the rows of H x for arbitrary row ranges (unequal shards, a single row, the empty range)
    assemble to the oracle's H x."""
    from paper_1204_3425_b200 import sharded
    ref = RefModel(ns, nu, nd, bonds, 1.0, 4.0)
    m = hb.hubbard_create(ns, nu, nd, bonds, 1.0, 4.0, dtype)
    x, x_np = start_vector(123, m.dim, dtype)
    y_ref = ref.apply(x_np)
    for world in (1, 3, 8):
        y = torch.full_like(x, float("nan"))
        for r0, r1 in sharded.row_partition(m.dim_up, world):
            yr = torch.full(((r1 - r0) * m.dim_dn,), float("nan"), dtype=x.dtype, device=x.device)
            m.hubbard_apply_rows(x, yr, r0, r1)
            y[r0 * m.dim_dn:r1 * m.dim_dn] = yr
        torch.cuda.synchronize()
        assert rel_max_err(y, y_ref) <= TOL_HV[dtype]
    with pytest.raises(hb.HubbardError):
        m.hubbard_apply_rows(x, y, 2, m.dim_up + 1)


def _run_virtual_ranks(m, world, v0, iters, tau):
    """Drives `world` instances of sharded_lanczos in lock-step on one GPU: each exchange step is resolved when every
    rank has reached it (threads + barriers; the kernels of different ranks simply queue on the stream)."""
    import threading
    from paper_1204_3425_b200 import sharded
    parts = sharded.row_partition(m.dim_up, world)
    bar = threading.Barrier(world)
    slots = {"gather": [None] * world, "reduce": [None] * world}
    results = [None] * world

    class Coll:
        def __init__(self, rank):
            self.rank = rank

        def all_gather_rows(self, shard, parts_, dim_dn, out_full):
            slots["gather"][self.rank] = shard
            bar.wait()
            for r, (r0, r1) in enumerate(parts_):
                out_full[r0 * dim_dn:r1 * dim_dn].copy_(slots["gather"][r])
            torch.cuda.synchronize()
            bar.wait()
            return out_full

        def all_reduce_sum(self, scalar):
            slots["reduce"][self.rank] = float(scalar.item())
            bar.wait()
            tot = sum(slots["reduce"])            # same order on every rank
            bar.wait()
            return tot

    def work(rank):
        torch.cuda.set_device(0)
        r0, r1 = parts[rank]
        ops = sharded.LibraryOps(models[rank], dev())
        results[rank] = sharded.sharded_lanczos(ops, Coll(rank), rank, world, m.dim_up, m.dim_dn,
                                                v0[r0 * m.dim_dn:r1 * m.dim_dn].clone(), iters, tau)

    models = [m] + [None] * (world - 1)
    return models, work, results


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_sharded_lanczos_virtual_ranks_vs_oracle(dtype):
    """The row-sharded Lanczos with the LIBRARY's kernels behind it (hubbard_apply_rows, lanczos_shard_update), three
    ranks' shards driven in lock-step on one GPU, against Algorithm 1 on the oracle: coefficient prefix, E_0, and the
    same numbers on every rank.  (The multi-process exchange itself is covered on CPU: tests/test_sharded_cpu.py.)"""
    import threading
    c = CONFIGS["C2"]
    world, iters = 3, 60
    ref = RefModel(c.n_sites, c.n_up, c.n_dn, c.bonds, c.t, 4.0)
    v0, v0_np = start_vector(c.seed, c.dim, dtype)
    m0 = hb.hubbard_create(c.n_sites, c.n_up, c.n_dn, c.bonds, c.t, 4.0, dtype)
    models, work, results = _run_virtual_ranks(m0, world, v0, iters, 1e-10 if dtype == "f64" else 1e-5)
    for r in range(1, world):                     # one model per rank, as on several GPUs
        models[r] = hb.hubbard_create(c.n_sites, c.n_up, c.n_dn, c.bonds, c.t, 4.0, dtype)
    threads = [threading.Thread(target=work, args=(r,)) for r in range(world)]
    for t in threads:
        t.start()
    for t in threads:
        t.join(timeout=600)
    assert all(r is not None for r in results)
    a_ref, b_ref = lr.lanczos(ref.apply, v0_np, iters)
    n = 30
    tol_c = 1e-10 if dtype == "f64" else 1e-5
    for alpha, beta in results:
        alpha, beta = np.array(alpha), np.array(beta)
        assert len(alpha) == iters
        assert np.max(np.abs(alpha[:n] - a_ref[:n]) / np.maximum(1.0, np.abs(a_ref[:n]))) <= tol_c
        assert np.max(np.abs(beta[:n] - b_ref[:n]) / np.maximum(1.0, np.abs(b_ref[:n]))) <= tol_c
        e_ref = lr.ground_energy(a_ref, b_ref)
        assert abs(hb.lanczos_ground_energy(alpha, beta) - e_ref) <= TOL_E0[dtype] * abs(e_ref)
    assert results[0] == results[1] == results[2]
