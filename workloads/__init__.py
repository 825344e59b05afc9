"""Seeded synthetic inputs shared by the oracle tests, the CUDA parity tests and
bench.py.  Holds none of the NNP arithmetic (only parameter grids, random
numbers and the rejection test of the position generator)."""
from __future__ import annotations

from dataclasses import dataclass

from .model import KIND_ANGULAR, KIND_RADIAL, SF_DTYPE, Model, make_model, sf_table
from .metal import A_NI, RC_NI, make_fcc
from .water import (ELEMENTS, TYPE_H, TYPE_O, WaterSystem, box_length, displacement,
                    make_cluster, make_water)


@dataclass(frozen=True)
class Config:
    name: str
    n_molecules: int
    wide: bool
    calls: int
    seed_pos: int
    seed_weights: int
    seed_disp: int | None = None
    kind: str = "water"            # "water" (BASELINE.json configs) or "metal" (fcc, n_molecules = cells per side)

    @property
    def n_atoms(self) -> int:
        return 3 * self.n_molecules if self.kind == "water" else 4 * self.n_molecules ** 3


# BASELINE.json configs[0..4]; seeds from SURVEY.md 8(d)
CONFIGS = (
    Config("tiny288", 96, False, 1, 200200054, 200200154),
    Config("small24k", 8192, False, 100, 200200055, 200200154, 200200255),
    Config("medium196k", 65536, False, 10, 200200056, 200200154),
    Config("large2M", 699051, False, 5, 200200057, 200200154),
    Config("wide196k", 65536, True, 10, 200200056, 200200158),
    # not a BASELINE.json config: SURVEY.md 8(f)2, Ni-like single-element metal, 72^3 fcc cells = 1,492,992 atoms
    Config("nickel1.5M", 72, False, 5, 200200060, 200200160, None, "metal"),
)


def get_config(k) -> Config:
    if isinstance(k, int):
        return CONFIGS[k]
    for c in CONFIGS:
        if c.name == k:
            return c
    raise KeyError(k)


def build(cfg: Config):
    """-> (WaterSystem, Model) for a config."""
    if cfg.kind == "metal":     # 8 radial + 12 angular SFs on one element, network 20-30-30-1 ("~30 x 2")
        return (make_fcc(cfg.n_molecules, cfg.seed_pos),
                make_model(False, cfg.seed_weights, rc=RC_NI, elements=("Ni",), hidden=(30, 30)))
    return make_water(cfg.n_molecules, cfg.seed_pos), make_model(cfg.wide, cfg.seed_weights)
