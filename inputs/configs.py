"""The five workload configurations of BASELINE.json (`configs[0..4]`), as
plain data: lattice, filling, couplings, Lanczos iteration count and the seed
of the start vector.  No method arithmetic lives here.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from math import comb

from .lattices import ring_bonds, torus_bonds

SEED_BASE = 12043425


@dataclass(frozen=True)
class Config:
    name: str
    lattice: str
    n_sites: int
    n_up: int
    n_dn: int
    bonds: tuple
    t: float
    U_values: tuple
    dtypes: tuple
    iters: int
    seed: int
    note: str = ""

    @property
    def dim_up(self) -> int:
        return comb(self.n_sites, self.n_up)

    @property
    def dim_dn(self) -> int:
        return comb(self.n_sites, self.n_dn)

    @property
    def dim(self) -> int:
        return self.dim_up * self.dim_dn


CONFIGS = {
    "C1": Config("C1", "ring8", 8, 4, 4, tuple(ring_bonds(8)), 1.0, (4.0,), ("f64",), 100,
                 SEED_BASE + 1, "BASELINE.json configs[0]"),
    "C2": Config("C2", "ring12", 12, 6, 6, tuple(ring_bonds(12)), 1.0, (4.0, 8.0), ("f32", "f64"), 200,
                 SEED_BASE + 2, "BASELINE.json configs[1]"),
    "C3": Config("C3", "torus4x4", 16, 5, 5, tuple(torus_bonds(4, 4)), 1.0, (8.0,), ("f32", "f64"), 200,
                 SEED_BASE + 3, "BASELINE.json configs[2]"),
    "C4": Config("C4", "torus4x4", 16, 8, 8, tuple(torus_bonds(4, 4)), 1.0, (4.0, 8.0), ("f32", "f64"), 200,
                 SEED_BASE + 4, "BASELINE.json configs[3] (headline: 4x4 half-filled)"),
    "C5": Config("C5", "ring18", 18, 9, 9, tuple(ring_bonds(18)), 1.0, (4.0,), ("f32", "f64"), 100,
                 SEED_BASE + 5, "BASELINE.json configs[4]"),
}


def get_config(name: str) -> Config:
    return CONFIGS[name]
