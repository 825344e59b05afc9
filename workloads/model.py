"""Seeded synthetic NNP models: symmetry-function tables and network weights.

Data only (parameter grids and random weights); the functions that *use* these
parameters live in oracle/ (CPU) and in the CUDA library, separately.

Readings of BASELINE.json taken here:
  C8  base angular set = 12 per neighbour-element pair:
        eta=0.001: lambda in (+1,-1) x zeta in (1,2,4,16)   (8)
        eta=0.01 : lambda = +1      x zeta in (1,2,4,16)   (4)
  C9  wide set: 16 radial eta_k = 0.001*500**(k/15); angular
        eta in (0.001,0.003,0.01,0.03) x lambda in (+1,-1) x zeta in (1,2,4,16) (32)
  C10 base radial eta_k = 0.001*500**(k/7), k=0..7, Rs = 0
  C11 order inside G: radial block (neighbour element 0, then 1; eta ascending),
      then angular block (pairs (0,0),(0,1),(1,1); eta ascending; lambda=+1 then
      -1; zeta ascending)
  C12 weights AND biases ~ N(0, 1/fan_in) (variance), row-major W[out][in],
      softplus hidden layers, linear output.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

from . import rng

KIND_RADIAL = 2      # n2p2 numbering: type 2 = radial Gaussian
KIND_ANGULAR = 3     # type 3 = angular "narrow"

SF_DTYPE = np.dtype(
    [("central", "<i4"), ("kind", "<i4"), ("e1", "<i4"), ("e2", "<i4"),
     ("eta", "<f8"), ("rs", "<f8"), ("lam", "<f8"), ("zeta", "<f8")],
    align=True,
)
assert SF_DTYPE.itemsize == 48


@dataclass
class Model:
    elements: tuple            # element names, index = type id
    rc: float                  # cutoff radius (A)
    sf: np.ndarray             # SF_DTYPE[n_sf]; order per central element = order in G
    layer_sizes: list          # per element: [n_in, h1, ..., 1]
    weights: list              # per element: flat f64 [W1(out x in), b1, W2, b2, ..., W_last, b_last]
    name: str = ""
    n_sf_per_elem: list = field(default_factory=list)
    # model generality: per element (shift[n_sf], scale[n_sf]) with network input
    # x = scale * (G - shift), or None; hidden activation "softplus" (BASELINE.json) or "tanh"
    sf_scaling: list | None = None
    activation: str = "softplus"
    # per-SF cutoff radii in the order of `sf` (each <= rc), or None: one global rc
    sf_cutoffs: list | None = None


def radial_etas(n: int) -> np.ndarray:
    k = np.arange(n, dtype=np.float64)
    return 0.001 * 500.0 ** (k / (n - 1))


def angular_grid(wide: bool):
    zetas = (1.0, 2.0, 4.0, 16.0)
    out = []
    if not wide:
        for lam in (1.0, -1.0):
            for z in zetas:
                out.append((0.001, lam, z))
        for z in zetas:
            out.append((0.01, 1.0, z))
    else:
        for eta in (0.001, 0.003, 0.01, 0.03):
            for lam in (1.0, -1.0):
                for z in zetas:
                    out.append((eta, lam, z))
    return out


def sf_table(n_elem: int = 2, wide: bool = False) -> np.ndarray:
    n_rad = 16 if wide else 8
    etas = radial_etas(n_rad)
    ang = angular_grid(wide)
    rows = []
    for c in range(n_elem):
        for e1 in range(n_elem):
            for eta in etas:
                rows.append((c, KIND_RADIAL, e1, 0, eta, 0.0, 0.0, 0.0))
        for e1 in range(n_elem):
            for e2 in range(e1, n_elem):
                for (eta, lam, z) in ang:
                    rows.append((c, KIND_ANGULAR, e1, e2, eta, 0.0, lam, z))
    return np.array(rows, dtype=SF_DTYPE)


def mlp_weights(layer_sizes, seed: int, elem: int) -> np.ndarray:
    """Flat [W1, b1, W2, b2, ...]; every entry N(0, 1/fan_in)."""
    key = rng.stream_key(seed, 0x776774, elem)  # "wgt"
    parts = []
    ctr = 0
    for l in range(len(layer_sizes) - 1):
        fan_in, fan_out = layer_sizes[l], layer_sizes[l + 1]
        n = fan_out * fan_in + fan_out
        c = np.arange(ctr, ctr + n, dtype=np.uint64)
        ctr += n
        parts.append(rng.normal(key, c) / np.sqrt(float(fan_in)))
    return np.concatenate(parts)


def make_model(wide: bool = False, seed: int | None = None, rc: float = 6.0,
               elements=("H", "O"), hidden=None) -> Model:
    n_elem = len(elements)
    sf = sf_table(n_elem, wide)
    if seed is None:
        seed = 200200158 if wide else 200200154
    if hidden is None:
        hidden = (64, 64) if wide else (25, 25)
    n_sf_per_elem = [int(np.sum(sf["central"] == c)) for c in range(n_elem)]
    layer_sizes = [[n_sf_per_elem[c], *hidden, 1] for c in range(n_elem)]
    weights = [mlp_weights(layer_sizes[c], seed, c) for c in range(n_elem)]
    return Model(elements=tuple(elements), rc=rc, sf=sf, layer_sizes=layer_sizes,
                 weights=weights, name="wide128" if wide else "base52",
                 n_sf_per_elem=n_sf_per_elem)
