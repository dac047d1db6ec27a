"""ORACLE, tier 1 binding (TEST INFRASTRUCTURE ONLY): ctypes access to
oracle/hubbard_ref.c, built with gcc on first use.  See that file's header for
what it is and what pins it.  Nothing under paper_1204_3425_b200/ imports this.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "hubbard_ref.c"
_LIB = _HERE / "libhubbard_ref.so"
_lib = None


def build(force: bool = False) -> Path:
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        cmd = ["gcc", "-O3", "-fopenmp", "-fPIC", "-shared", "-std=c11",
               "-o", str(_LIB), str(_SRC), "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(str(_LIB))
        _lib.ref_basis.restype = C.c_int64
        _lib.ref_hops_csr.restype = C.c_int64
        _lib.ref_lanczos.restype = C.c_int
        _lib.ref_max_threads.restype = C.c_int
    return _lib


def _p(a, ty):
    return a.ctypes.data_as(C.POINTER(ty))


def max_threads() -> int:
    return int(_load().ref_max_threads())


class RefModel:
    """Tier-1 model: basis lists + CSR hop tables + matrix-free H*v (fp64)."""

    def __init__(self, n_sites: int, n_up: int, n_dn: int, bonds, t: float, U: float):
        lib = _load()
        self.n_sites, self.n_up, self.n_dn = n_sites, n_up, n_dn
        self.t, self.U = float(t), float(U)
        self.bonds = np.ascontiguousarray(np.array(list(bonds), dtype=np.int32).reshape(-1, 2))
        nb = len(self.bonds)
        self.states, self.csr = {}, {}
        for spin, n_el, n_left in ((0, n_up, 0), (1, n_dn, n_up)):
            n = lib.ref_basis(n_sites, n_el, None, C.c_int64(0))
            st = np.empty(n, dtype=np.uint32)
            lib.ref_basis(n_sites, n_el, _p(st, C.c_uint32), C.c_int64(n))
            cap = max(1, n * 2 * max(1, nb))
            rp = np.empty(n + 1, dtype=np.int64)
            cj = np.empty(cap, dtype=np.int32)
            cv = np.empty(cap, dtype=np.float64)
            nnz = lib.ref_hops_csr(n_sites, n_el, n_left, _p(self.bonds, C.c_int32), nb, C.c_double(self.t),
                                   _p(st, C.c_uint32), C.c_int64(n), _p(rp, C.c_int64), _p(cj, C.c_int32),
                                   _p(cv, C.c_double), C.c_int64(cap))
            assert nnz >= 0
            self.states[spin] = st
            self.csr[spin] = (rp, cj[:nnz].copy(), cv[:nnz].copy())
        self.dim_up, self.dim_dn = len(self.states[0]), len(self.states[1])
        self.dim = self.dim_up * self.dim_dn

    def hop_rows(self, spin: int):
        """Canonical form: list over rows of [(col, value), ...] sorted by col."""
        rp, cj, cv = self.csr[spin]
        return [[(int(cj[k]), float(cv[k])) for k in range(rp[r], rp[r + 1])] for r in range(len(rp) - 1)]

    def hop_ell(self, spin: int):
        """Canonical ELL form (row-major n x width, sorted by column, padding
        col = -1 / val = 0) — the layout `hubbard_get_hops` returns."""
        rp, cj, cv = self.csr[spin]
        n = len(rp) - 1
        cnt = np.diff(rp)
        width = int(cnt.max()) if n else 0
        cols = np.full((n, width), -1, dtype=np.int32)
        vals = np.zeros((n, width), dtype=np.float64)
        k = np.arange(len(cj)) - np.repeat(rp[:-1], cnt)
        r = np.repeat(np.arange(n), cnt)
        cols[r, k] = cj
        vals[r, k] = cv
        return width, cols, vals

    def _args(self):
        a = []
        for spin in (0, 1):
            rp, cj, cv = self.csr[spin]
            a += [_p(rp, C.c_int64), _p(cj, C.c_int32), _p(cv, C.c_double)]
        return a

    def apply(self, x: np.ndarray, n_threads: int = 0, U: float | None = None) -> np.ndarray:
        x = np.ascontiguousarray(x, dtype=np.float64)
        assert x.size == self.dim
        y = np.empty(self.dim, dtype=np.float64)
        _load().ref_apply(C.c_int64(self.dim_up), C.c_int64(self.dim_dn),
                          _p(self.states[0], C.c_uint32), _p(self.states[1], C.c_uint32), *self._args(),
                          C.c_double(self.U if U is None else U), _p(x, C.c_double), _p(y, C.c_double),
                          C.c_int(n_threads))
        return y

    def lanczos_two_vector(self, v0: np.ndarray, m: int, tau: float = 1e-10, n_threads: int = 0):
        """The paper's CPU comparator (Algorithm 1 + eq. 13), for timing and as
        a cross-check of oracle/lanczos_ref.py."""
        f = np.array(v0, dtype=np.float64, copy=True)
        g = np.empty_like(f)
        h = np.empty_like(f)
        alpha = np.zeros(m)
        beta = np.zeros(m)
        done = _load().ref_lanczos(C.c_int64(self.dim_up), C.c_int64(self.dim_dn),
                                   _p(self.states[0], C.c_uint32), _p(self.states[1], C.c_uint32), *self._args(),
                                   C.c_double(self.U), _p(f, C.c_double), _p(g, C.c_double), _p(h, C.c_double),
                                   C.c_int(m), C.c_double(tau), _p(alpha, C.c_double), _p(beta, C.c_double),
                                   C.c_int(n_threads))
        return alpha[:done], beta[:done]
