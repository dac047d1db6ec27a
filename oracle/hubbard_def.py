"""ORACLE, tier 0 (TEST INFRASTRUCTURE ONLY — never imported by the product).

The Hubbard Hamiltonian built element by element from its definition,
PAPER.md:23-25 (eq. 1-3):

    H = -t sum_<ij> sum_sigma (c+_{i,sigma} c_{j,sigma} + h.c.) + U sum_i n_{i,up} n_{i,dn}

in the basis of PAPER.md:41-47 (eq. 4): a basis ket is a string of creation
operators acting on the empty lattice |O>, all spin-up operators to the left
of all spin-down operators, site indices ascending from left to right.  Every
operator of H is applied LITERALLY to that string, one anticommutation
(eq. 3) at a time, counting one minus sign per exchange.  There is no
Kronecker split, no "electrons hopped over" shortcut, no table shared with the
CUDA path.  Slow on purpose: pure-Python loops, usable up to a few thousand
basis states densely, and row by row (`row_of_H`) at any size.

Ordering of basis kets (eq. 7): J = i_up * C(N_s, N_dn) + i_dn
with i_sigma the position of the spin's bit pattern (bit k = site k occupied,
PAPER.md:56-61) in the ascending list of all N_s-bit numbers with N_sigma bits
set.  The list is obtained by enumerating ALL 2^N_s numbers and keeping those
with the right popcount — no ranking formula.

Pins (tests/test_oracle_pins.py, all `-m "not gpu"`): PAPER.md Table 1 and
eq. 8-10 (tests/golden/paper_table1.txt, paper_matrix_elements.txt), eq. 5
dimensions, exact Hermiticity, the 2-site closed form, U=0 free-fermion
energies, t=0 energies, dense brute force against an independent
second-quantisation construction (Jordan-Wigner matrices) on <= 6 sites.
"""
from __future__ import annotations

import numpy as np

UP, DN = 0, 1


# ---------------------------------------------------------------------------
# basis
# ---------------------------------------------------------------------------
def sector_states(n_sites: int, n_el: int) -> list[int]:
    """Ascending list of all n_sites-bit numbers with n_el bits set."""
    return [s for s in range(1 << n_sites) if bin(s).count("1") == n_el]


def ket_from_bits(up_bits: int, dn_bits: int, n_sites: int) -> tuple:
    """Canonical operator string of eq. (4): ((spin, site), ...), up first,
    sites ascending."""
    ups = [(UP, k) for k in range(n_sites) if (up_bits >> k) & 1]
    dns = [(DN, k) for k in range(n_sites) if (dn_bits >> k) & 1]
    return tuple(ups + dns)


def bits_from_ket(ket: tuple) -> tuple[int, int]:
    up = dn = 0
    for spin, site in ket:
        if spin == UP:
            up |= 1 << site
        else:
            dn |= 1 << site
    return up, dn


# ---------------------------------------------------------------------------
# literal operator algebra (eq. 3)
# ---------------------------------------------------------------------------
def annihilate(ket: tuple, op: tuple):
    """c_op applied to  c+_{k0} c+_{k1} ... |O>.

    c_op is moved to the right one creation operator at a time.  Passing a
    different operator costs a factor -1 ({c, c+'} = 0).  Meeting its own
    creation operator, c c+ = 1 - c+ c: the '1' term leaves the rest of the
    string untouched; the 'c+ c' term keeps moving right and finally hits
    c|O> = 0 (a canonical string holds each operator at most once).
    Returns (sign, new_ket) or None for the zero vector.
    """
    sign = 1
    for pos, k in enumerate(ket):
        if k == op:
            return sign, ket[:pos] + ket[pos + 1:]
        sign = -sign
    return None  # c|O> = 0


def create(ket: tuple, op: tuple):
    """c+_op applied to a canonical string: written at the far left, then
    moved right by adjacent exchanges ({c+, c+'} = 0: -1 each) until the
    string is again in the canonical order (spin, site) ascending.
    (c+)^2 = 0.  Returns (sign, new_ket) or None."""
    if op in ket:
        return None
    sign = 1
    pos = 0
    while pos < len(ket) and ket[pos] < op:  # tuple order = (spin, site): up < dn, sites ascending
        sign = -sign
        pos += 1
    return sign, ket[:pos] + (op,) + ket[pos:]


def apply_H_to_ket(ket: tuple, bonds, t: float, U: float) -> dict:
    """H|ket> as {ket': coefficient}, eq. (2) term by term."""
    out: dict = {}

    def add(k, c):
        out[k] = out.get(k, 0.0) + c

    # hopping: -t (c+_i c_j + c+_j c_i) for both spins
    for (i, j) in bonds:
        for spin in (UP, DN):
            for (dst, src) in ((i, j), (j, i)):
                r = annihilate(ket, (spin, src))
                if r is None:
                    continue
                s1, k1 = r
                r = create(k1, (spin, dst))
                if r is None:
                    continue
                s2, k2 = r
                add(k2, -t * s1 * s2)
    # interaction: U n_{i,up} n_{i,dn}, n = c+ c, applied right to left
    if U != 0.0:
        sites = sorted({s for b in bonds for s in b} | {site for _, site in ket})
        for i in sites:
            k, sgn = ket, 1
            ok = True
            for op in ((DN, i), (UP, i)):       # n_dn first (rightmost factor), then n_up
                r = annihilate(k, op)
                if r is None:
                    ok = False
                    break
                s1, k1 = r
                r = create(k1, op)
                if r is None:
                    ok = False
                    break
                s2, k = r
                sgn *= s1 * s2
            if ok:
                add(k, U * sgn)
    return {k: c for k, c in out.items() if c != 0.0}


# ---------------------------------------------------------------------------
# the sector and its dense matrix
# ---------------------------------------------------------------------------
class Sector:
    """Fixed (N_s, N_up, N_dn) subspace with the paper's labelling J."""

    def __init__(self, n_sites: int, n_up: int, n_dn: int):
        self.n_sites, self.n_up, self.n_dn = n_sites, n_up, n_dn
        self.states_up = sector_states(n_sites, n_up)
        self.states_dn = sector_states(n_sites, n_dn)
        self.dim_up, self.dim_dn = len(self.states_up), len(self.states_dn)
        self.dim = self.dim_up * self.dim_dn
        self.pos_up = {s: i for i, s in enumerate(self.states_up)}
        self.pos_dn = {s: i for i, s in enumerate(self.states_dn)}

    def J_of_bits(self, up_bits: int, dn_bits: int) -> int:
        return self.pos_up[up_bits] * self.dim_dn + self.pos_dn[dn_bits]  # eq. (7)

    def bits_of_J(self, J: int) -> tuple[int, int]:
        return self.states_up[J // self.dim_dn], self.states_dn[J % self.dim_dn]

    def ket_of_J(self, J: int) -> tuple:
        u, d = self.bits_of_J(J)
        return ket_from_bits(u, d, self.n_sites)

    def J_of_ket(self, ket: tuple) -> int:
        return self.J_of_bits(*bits_from_ket(ket))


def column_of_H(sec: Sector, J: int, bonds, t: float, U: float) -> dict:
    """{J': <J'|H|J>}: the J-th column of H from the definition."""
    res = apply_H_to_ket(sec.ket_of_J(J), bonds, t, U)
    return {sec.J_of_ket(k): c for k, c in res.items()}


def row_of_H(sec: Sector, J: int, bonds, t: float, U: float) -> dict:
    """{J': <J|H|J'>}.  H is real symmetric (hermitian with real t, U;
    pinned by the exact-Hermiticity test), so row J equals column J."""
    return column_of_H(sec, J, bonds, t, U)


def dense_hamiltonian(n_sites: int, n_up: int, n_dn: int, bonds, t: float, U: float) -> np.ndarray:
    sec = Sector(n_sites, n_up, n_dn)
    H = np.zeros((sec.dim, sec.dim), dtype=np.float64)
    for J in range(sec.dim):
        for Jp, c in column_of_H(sec, J, bonds, t, U).items():
            H[Jp, J] += c
    return H


def sampled_Hv(sec: Sector, bonds, t: float, U: float, sample_J, v_of) -> np.ndarray:
    """(H v)[J] for each J in sample_J, with v given as a function
    v_of(index_array) -> values (e.g. the counter-based start vector), so the
    full vector is never materialised (pin P10)."""
    out = np.empty(len(sample_J), dtype=np.float64)
    for n, J in enumerate(sample_J):
        row = row_of_H(sec, int(J), bonds, t, U)
        cols = np.fromiter(row.keys(), dtype=np.int64, count=len(row))
        vals = np.fromiter(row.values(), dtype=np.float64, count=len(row))
        order = np.argsort(cols)
        out[n] = float(np.dot(vals[order], v_of(cols[order]))) if len(cols) else 0.0
    return out


# ---------------------------------------------------------------------------
# per-spin hopping tables in canonical form (for the bit-exact table parity)
# ---------------------------------------------------------------------------
def hop_table(n_sites: int, n_up: int, n_dn: int, spin: int, bonds, t: float, other_bits: int | None = None):
    """Per-spin hopping matrix H_sigma of eq. (14) from the
    definition: <i'|H_hop|i> between kets that differ only in the spin-`spin`
    pattern, with the other spin frozen in `other_bits` (default: its lowest
    pattern).  Returned in canonical form: list over rows i' of sorted
    [(col, value), ...] with duplicates merged.

    That the result does not depend on `other_bits` (no cross-spin sign,
    DESIGN.md reading Q3) is a tested property, not an assumption.
    """
    sec = Sector(n_sites, n_up, n_dn)
    mine = sec.states_up if spin == UP else sec.states_dn
    pos = sec.pos_up if spin == UP else sec.pos_dn
    others = sec.states_dn if spin == UP else sec.states_up
    if other_bits is None:
        other_bits = others[0]
    rows: list[dict] = [dict() for _ in mine]
    for i, s in enumerate(mine):
        ket = ket_from_bits(s, other_bits, n_sites) if spin == UP else ket_from_bits(other_bits, s, n_sites)
        for k2, c in apply_H_to_ket(ket, bonds, t, 0.0).items():
            u, d = bits_from_ket(k2)
            if spin == UP and d == other_bits:
                rows[pos[u]][i] = rows[pos[u]].get(i, 0.0) + c
            elif spin == DN and u == other_bits:
                rows[pos[d]][i] = rows[pos[d]].get(i, 0.0) + c
    return [sorted((c, v) for c, v in r.items() if v != 0.0) for r in rows]
