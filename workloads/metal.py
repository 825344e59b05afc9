"""Seeded synthetic single-element metallic system shaped like the paper's Ni workload (Ni NNP
with a 3.9 A cutoff; L96: ~1.5 M atoms): an fcc lattice (a = 3.52 A) with Gaussian thermal displacements.
SURVEY.md 8(f)2.  No NNP arithmetic here; the mlearn Ni model is not in the container, so the weights are
synthetic (workloads.model.make_model with one element)."""
from __future__ import annotations

import numpy as np

from . import rng
from .water import WaterSystem

A_NI = 3.52
RC_NI = 3.9


def make_fcc(n_cells: int, seed: int, a: float = A_NI, sigma: float = 0.08) -> WaterSystem:
    """4 n_cells^3 atoms of element 0 in a cubic box of side n_cells * a, displaced by N(0, sigma^2) per component.
    With rc = 3.9 A every atom sees the first two fcc shells: 18 neighbours, 153 (j,k) pairs, 60 triangles."""
    base = np.array([[0.0, 0.0, 0.0], [0.5, 0.5, 0.0], [0.5, 0.0, 0.5], [0.0, 0.5, 0.5]])
    g = np.stack(np.meshgrid(*[np.arange(n_cells, dtype=np.float64)] * 3, indexing="ij"), -1).reshape(-1, 1, 3)
    pos = ((g + base[None]).reshape(-1, 3)) * a
    n = pos.shape[0]
    key = rng.stream_key(seed, 0x666363)  # "fcc"
    pos = pos + sigma * rng.normal(key, np.arange(3 * n, dtype=np.uint64)).reshape(n, 3)
    L = n_cells * a
    pos -= L * np.floor(pos / L)
    np.minimum(pos, np.nextafter(L, 0.0), out=pos)
    return WaterSystem(pos=pos, types=np.zeros(n, dtype=np.int32), box=np.array([L, L, L]), seed=seed)
