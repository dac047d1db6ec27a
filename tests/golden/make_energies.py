#!/usr/bin/env python
"""Writes tests/golden/oracle_energies.txt: Lanczos coefficients and ground-state
energies of the five BASELINE.json configurations computed ONLY with the oracle
(oracle/lanczos_ref.py = Algorithm 1 verbatim, on the tier-1
matrix-free H*v of oracle/hubbard_ref.c) and the seeded start vectors of
inputs/.  Nothing from paper_1204_3425_b200/ is imported or executed.

    python tests/golden/make_energies.py [C1 C2 C3 C4 C5 ...]      (default: C1 C2 C3 C4)

The GPU parity tests read the file (tests/test_gpu_parity.py) because the
full-length oracle runs are too slow for the test suite itself: C4 takes about
a quarter of an hour per U on 8 host cores, C5 needs ~40-57 GB of host RAM.

Record format, one per (config, U), whitespace separated:
    case  <name> <U> <iters> <seed>
    E0    <lambda_min(T_iters)>           numpy eigvalsh on the explicit T_m
    alpha <first n_prefix a_j>            17 significant digits
    beta  <first n_prefix b_{j+1}>
C5 stores the first 2 iterations only (a_1, b_2, a_2, b_3), computed in place
with two resident host vectors of 18.9 GB.
"""
from __future__ import annotations

import sys
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parents[2]
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

from inputs import CONFIGS, g_uniform, start_vector_np  # noqa: E402
from oracle import lanczos_ref as lr  # noqa: E402
from oracle.ref import RefModel  # noqa: E402

OUT = Path(__file__).resolve().parent / "oracle_energies.txt"
N_PREFIX = 50


def fmt(x):
    return " ".join(f"{v:.17g}" for v in x)


def full_case(name, U):
    c = CONFIGS[name]
    ref = RefModel(c.n_sites, c.n_up, c.n_dn, c.bonds, c.t, U)
    v0 = start_vector_np(c.seed, c.dim)
    v0 /= np.sqrt(np.dot(v0, v0))
    t0 = time.time()
    a, b = lr.lanczos(ref.apply, v0, c.iters)
    e0 = lr.ground_energy(a, b)
    print(f"{name} U={U}: {len(a)} iterations, E0 = {e0:.15g}  ({time.time() - t0:.0f} s)", file=sys.stderr)
    return [f"case  {name} {U:g} {len(a)} {c.seed}", f"E0    {e0:.17g}", f"alpha {fmt(a[:N_PREFIX])}",
            f"beta  {fmt(b[:N_PREFIX])}"]


def chunked(n, step=1 << 26):
    for lo in range(0, n, step):
        yield slice(lo, min(n, lo + step))


def cdot(x, y):
    return float(sum(np.dot(x[s], y[s]) for s in chunked(x.size)))


def c5_case(U):
    """Algorithm 1 lines 4-11 written out for the first two iterations with
    in-place chunked vector operations and two resident host vectors: f_1 is
    regenerated chunk by chunk from the counter-based generator where line 4 of
    iteration 2 needs it (b_2 f_1)."""
    c = CONFIGS["C5"]
    ref = RefModel(c.n_sites, c.n_up, c.n_dn, c.bonds, c.t, U)
    t0 = time.time()
    f = start_vector_np(c.seed, c.dim)
    nrm = np.sqrt(cdot(f, f))
    for s in chunked(f.size):
        f[s] /= nrm                             # f_1
    alpha, beta = [], []
    # iteration 1: b_1 = 0, f_0 = 0 (lines 1-2)
    q = ref.apply(f)                            # line 4
    a = cdot(q, f)                              # line 5
    for s in chunked(f.size):
        q[s] -= a * f[s]                        # line 6
    b = np.sqrt(cdot(q, q))                     # line 7
    alpha.append(a); beta.append(b)
    print(f"C5 U={U}: a_1 = {a:.15g}, b_2 = {b:.15g}  ({time.time() - t0:.0f} s)", file=sys.stderr)
    for s in chunked(f.size):
        q[s] /= b                               # line 11: f_2
    del f
    f = q
    # iteration 2
    q = ref.apply(f)
    for s in chunked(f.size):
        f1 = g_uniform(c.seed, np.arange(s.start, s.stop, dtype=np.uint64)) / nrm
        q[s] -= b * f1                          # line 4
    a = cdot(q, f)
    for s in chunked(f.size):
        q[s] -= a * f[s]
    b = np.sqrt(cdot(q, q))
    alpha.append(a); beta.append(b)
    print(f"C5 U={U}: a_2 = {a:.15g}, b_3 = {b:.15g}  ({time.time() - t0:.0f} s)", file=sys.stderr)
    return [f"case  C5 {U:g} 2 {c.seed}", "E0    nan", f"alpha {fmt(alpha)}", f"beta  {fmt(beta)}"]


def main():
    names = sys.argv[1:] or ["C1", "C2", "C3", "C4"]
    records = {}
    if OUT.exists():                            # keep the records of configurations not recomputed now
        cur = None
        for line in OUT.read_text().splitlines():
            if line.startswith("case"):
                cur = tuple(line.split()[1:3])
                records[cur] = []
            if cur is not None and line and not line.startswith("#"):
                records[cur].append(line)
    for name in names:
        for U in CONFIGS[name].U_values:
            rec = c5_case(U) if name == "C5" else full_case(name, U)
            records[(name, f"{U:g}")] = rec
            header = ["# Written by tests/golden/make_energies.py (oracle only: Algorithm 1, PAPER.md:116-144, on",
                      "# oracle/hubbard_ref.c's H*v; start vector inputs.start_vector_np(seed), normalised, fp64).",
                      "# case <config> <U> <iterations> <seed> / E0 = lambda_min(T_m) / first coefficients."]
            body = [l for key in sorted(records) for l in records[key]]
            OUT.write_text("\n".join(header + body) + "\n")


if __name__ == "__main__":
    main()
