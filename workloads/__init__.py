"""Seeded synthetic inputs shared by the oracle tests, the CUDA parity tests and
bench.py.  Holds none of the NNP arithmetic (only parameter grids, random
numbers and the rejection test of the position generator)."""
from __future__ import annotations

from dataclasses import dataclass

from .model import KIND_ANGULAR, KIND_RADIAL, SF_DTYPE, Model, make_model, sf_table
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

    @property
    def n_atoms(self) -> int:
        return 3 * self.n_molecules


# BASELINE.json configs[0..4]; seeds from SURVEY.md 8(d)
CONFIGS = (
    Config("tiny288", 96, False, 1, 200200054, 200200154),
    Config("small24k", 8192, False, 100, 200200055, 200200154, 200200255),
    Config("medium196k", 65536, False, 10, 200200056, 200200154),
    Config("large2M", 699051, False, 5, 200200057, 200200154),
    Config("wide196k", 65536, True, 10, 200200056, 200200158),
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
    return make_water(cfg.n_molecules, cfg.seed_pos), make_model(cfg.wide, cfg.seed_weights)
