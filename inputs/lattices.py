"""Bond lists of the paper's workloads (§5: 1D periodic rings at
half filling and the 4x4 periodic square lattice).

A bond list is a list of undirected site pairs, each neighbour pair listed
once; both hop directions are implied by the "+ h.c." of eq. (2)
(PAPER.md:23).  Site labels are the bit positions of eq. (6).
"""
from __future__ import annotations


def ring_bonds(n_sites: int) -> list[tuple[int, int]]:
    """1D ring with periodic boundary: bonds (i, i+1 mod n_sites).

    The wrap bond is listed as (n_sites-1, 0) (reading Q5/Q6).
    n_sites = 2 would list the same pair twice; callers wanting the dimer pass
    [(0, 1)] themselves.
    """
    if n_sites < 2:
        return []
    return [(i, (i + 1) % n_sites) for i in range(n_sites)]


def chain_bonds(n_sites: int) -> list[tuple[int, int]]:
    """Open 1D chain: bonds (i, i+1)."""
    return [(i, i + 1) for i in range(n_sites - 1)]


def torus_bonds(lx: int, ly: int) -> list[tuple[int, int]]:
    """lx x ly square lattice, periodic in both directions, site = x + lx*y
    (reading Q7).  4x4 gives the 32 nearest-neighbour bonds of
    BASELINE.json configs 3 and 4.  A direction of extent 2 would duplicate
    its bonds and one of extent 1 would make self-bonds; both are skipped so
    every neighbour pair appears once.
    """
    bonds = []
    seen = set()
    for y in range(ly):
        for x in range(lx):
            s = x + lx * y
            for (xx, yy) in (((x + 1) % lx, y), (x, (y + 1) % ly)):
                t = xx + lx * yy
                key = (min(s, t), max(s, t))
                if s == t or key in seen:
                    continue
                seen.add(key)
                bonds.append((s, t))
    return bonds


def ladder_bonds(lx: int, ly: int) -> list[tuple[int, int]]:
    """Open lx x ly cluster (no periodic wraps), site = x + lx*y: a non-ring
    bond list for the small brute-force cases (e.g. the 2x3 cluster)."""
    bonds = []
    for y in range(ly):
        for x in range(lx):
            s = x + lx * y
            if x + 1 < lx:
                bonds.append((s, s + 1))
            if y + 1 < ly:
                bonds.append((s, s + lx))
    return bonds
