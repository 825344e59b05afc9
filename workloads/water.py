"""Seeded synthetic water-like systems (BASELINE.json configs[0..4]).

Shape of the paper's H2O workload (2 elements, ratio 2:1, ~6 A cutoff,
PAPER.md L70-72; ~2 M atoms on one GPU, L82).  The real n2p2 water model and
configurations are not available, so these stand in for them.

Recipe:
  * elements ("H", "O") -> type ids (0, 1); atoms are molecule-major O,H,H.
  * number density rho = 288 / 14.2**3 A^-3; cubic box L = (N / rho)**(1/3).
  * every coordinate iid uniform in [0, L).
  * rejection: an H atom closer than 0.9 A (minimum image) to ANY O atom is
    redrawn (new counter round) until no such pair is left.  O atoms never move,
    so the loop terminates; same-element pairs may be arbitrarily close.
  * displacements (configs[1]): before call t >= 1 every coordinate receives an
    extra N(0, sigma^2) kick, cumulative; positions are NOT re-wrapped here (the
    library wraps).

Only geometry bookkeeping lives here (a k-d tree for the rejection test); none
of the NNP arithmetic.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np
from scipy.spatial import cKDTree

from . import rng

RHO = 288.0 / 14.2 ** 3          # atoms / A^3  (configs[0]: 288 atoms, L = 14.2 A)
OH_MIN = 0.9                     # A
TYPE_H, TYPE_O = 0, 1
ELEMENTS = ("H", "O")


@dataclass
class WaterSystem:
    pos: np.ndarray      # [N][3] float64, A
    types: np.ndarray    # [N] int32 (0 = H, 1 = O)
    box: np.ndarray      # [3] float64, orthorhombic lengths, origin 0
    seed: int

    @property
    def n_atoms(self) -> int:
        return int(self.pos.shape[0])


def box_length(n_atoms: int) -> float:
    if n_atoms == 288:
        return 14.2
    return float((n_atoms / RHO) ** (1.0 / 3.0))


def _draw(key: int, atom_ids: np.ndarray, round_id: int, L: float) -> np.ndarray:
    """Uniform positions for the given atoms at redraw round `round_id`."""
    out = np.empty((atom_ids.size, 3), dtype=np.float64)
    kr = rng.stream_key(key, round_id)
    for c in range(3):
        out[:, c] = rng.uniform(kr, atom_ids.astype(np.uint64) * np.uint64(3) + np.uint64(c)) * L
    # (1 - 2^-53) * L can round up to L; keep strictly inside the box
    np.minimum(out, np.nextafter(L, 0.0), out=out)
    return out


def make_water(n_molecules: int, seed: int, L: float | None = None) -> WaterSystem:
    n = 3 * n_molecules
    if L is None:
        L = box_length(n)
    types = np.tile(np.array([TYPE_O, TYPE_H, TYPE_H], dtype=np.int32), n_molecules)
    key = rng.stream_key(seed, 0x706F73)  # "pos"
    ids = np.arange(n, dtype=np.int64)
    pos = _draw(key, ids, 0, L)
    o_idx = ids[types == TYPE_O]
    h_idx = ids[types == TYPE_H]
    tree_o = cKDTree(pos[o_idx], boxsize=L)
    pending = h_idx
    round_id = 0
    while pending.size:
        d, _ = tree_o.query(pos[pending], k=1, distance_upper_bound=OH_MIN)
        bad = pending[np.isfinite(d)]          # an O atom within 0.9 A exists
        if bad.size == 0:
            break
        round_id += 1
        if round_id > 200:
            raise RuntimeError("rejection sampling did not converge")
        pos[bad] = _draw(key, bad, round_id, L)
        pending = bad
    return WaterSystem(pos=pos, types=types, box=np.array([L, L, L], dtype=np.float64), seed=seed)


def displacement(n_atoms: int, seed: int, call: int, sigma: float = 0.01) -> np.ndarray:
    """N(0, sigma^2) kick added before call `call` (>= 1); cumulative across calls."""
    key = rng.stream_key(seed, 0x646973, call)  # "dis"
    c = np.arange(3 * n_atoms, dtype=np.uint64)
    return (sigma * rng.normal(key, c)).reshape(n_atoms, 3)


def make_cluster(n_atoms: int, seed: int, radius: float, L: float) -> WaterSystem:
    """Isolated blob of atoms (types O,H,H repeating) inside a big periodic box:
    used for arbitrary-rotation invariance tests (L > 2 * (2*radius + rc))."""
    key = rng.stream_key(seed, 0x636C75)
    ids = np.arange(n_atoms, dtype=np.uint64)
    p = np.empty((n_atoms, 3))
    for c in range(3):
        p[:, c] = (rng.uniform(key, ids * np.uint64(3) + np.uint64(c)) * 2.0 - 1.0) * radius
    p += L / 2.0
    types = np.tile(np.array([TYPE_O, TYPE_H, TYPE_H], dtype=np.int32), (n_atoms + 2) // 3)[:n_atoms]
    return WaterSystem(pos=p, types=types.copy(), box=np.array([L, L, L], dtype=np.float64), seed=seed)
