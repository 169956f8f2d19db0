"""Seeded synthetic input generators shared by the tests, bench.py and the oracle-side checks.

Holds NONE of the method's arithmetic: only random draws and shape bookkeeping, so that the
CUDA path and the CPU oracle can be fed identical inputs without sharing any code of the
method itself.
"""
from __future__ import annotations

import numpy as np


def site_legs(Lx, Ly, x, y):
    """Directions present at (x,y) in canonical order U,D,L,R."""
    legs = []
    if y > 0: legs.append("U")
    if y < Ly - 1: legs.append("D")
    if x > 0: legs.append("L")
    if x < Lx - 1: legs.append("R")
    return legs


def bond_id(Lx, Ly, x, y, d):
    nh = Ly * (Lx - 1)
    if d == "R": return y * (Lx - 1) + x
    if d == "L": return y * (Lx - 1) + x - 1
    if d == "D": return nh + y * Lx + x
    if d == "U": return nh + (y - 1) * Lx + x
    raise ValueError(d)


def n_bonds(Lx, Ly):
    return Ly * (Lx - 1) + (Ly - 1) * Lx


def synthetic_state(Lx, Ly, chi, seed_base=1000, decades=6.0):
    """SURVEY.md section 8(d) recipe (iii): bond e has dimension chi[e] (int or list), psi_v iid
    N(0,1) * size^-1/2 from seed seed_base + site, lambda_e[k] proportional to
    10^(-decades k/(chi-1)), normalised to unit 2-norm.  Returns (chi list, {site: packed
    column-major flat array}, [lambda_e])."""
    nb = n_bonds(Lx, Ly)
    chis = [int(chi)] * nb if np.isscalar(chi) else [int(c) for c in chi]
    psi = {}
    for y in range(Ly):
        for x in range(Lx):
            v = y * Lx + x
            dims = [chis[bond_id(Lx, Ly, x, y, d)] for d in site_legs(Lx, Ly, x, y)] + [4]
            size = int(np.prod(dims))
            rng = np.random.default_rng(seed_base + v)
            psi[v] = rng.standard_normal(size) / np.sqrt(size)
    lam = []
    for e in range(nb):
        c = chis[e]
        l = 10.0 ** (-decades * np.arange(c) / max(c - 1, 1))
        lam.append(l / np.linalg.norm(l))
    return chis, psi, lam


def normal_tensor(shape, seed):
    """iid N(0,1) flat fp64 array of prod(shape) elements (BASELINE config 3)."""
    return np.random.default_rng(seed).standard_normal(int(np.prod(shape)))
