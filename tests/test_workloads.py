"""The seeded input generators: determinism, shapes and the stated recipe."""
import numpy as np
from scipy.spatial import cKDTree

import workloads as W
from workloads import rng


def test_rng_is_counter_based():
    k = rng.stream_key(123, 4, 5)
    a = rng.uniform(k, np.arange(100, dtype=np.uint64))
    b = rng.uniform(k, np.arange(50, 100, dtype=np.uint64))
    assert np.array_equal(a[50:], b)
    assert rng.stream_key(123, 4, 5) != rng.stream_key(123, 5, 4)
    assert 0.0 <= a.min() and a.max() < 1.0
    # splitmix64 reference vector: first output for state 0 is 0xE220A8397B1DCDAF
    assert int(rng.bits(0, np.array([0], dtype=np.uint64))[0]) == 0xE220A8397B1DCDAF


def test_config0_recipe():
    sysm, model = W.build(W.CONFIGS[0])
    again, _ = W.build(W.CONFIGS[0])
    assert np.array_equal(sysm.pos, again.pos)
    assert sysm.n_atoms == 288 and sysm.box[0] == 14.2
    assert np.sum(sysm.types == W.TYPE_O) == 96 and np.sum(sysm.types == W.TYPE_H) == 192
    assert list(sysm.types[:6]) == [1, 0, 0, 1, 0, 0]
    assert sysm.pos.min() >= 0.0 and sysm.pos.max() < 14.2
    o = sysm.pos[sysm.types == W.TYPE_O]
    h = sysm.pos[sysm.types == W.TYPE_H]
    d, _ = cKDTree(o, boxsize=14.2).query(h, k=1)
    assert d.min() >= 0.9
    # model: 2*8 radial + 3*12 angular = 52 per central element; 52-25-25-1
    assert model.n_sf_per_elem == [52, 52]
    assert model.layer_sizes[0] == [52, 25, 25, 1]
    assert model.weights[0].shape == (52 * 25 + 25 + 25 * 25 + 25 + 25 + 1,)
    etas = model.sf[(model.sf["central"] == 0) & (model.sf["kind"] == 2) & (model.sf["e1"] == 0)]["eta"]
    assert abs(etas[0] - 0.001) < 1e-18 and abs(etas[-1] - 0.5) < 1e-15 and len(etas) == 8


def test_wide_model_shape():
    m = W.make_model(True)
    assert m.n_sf_per_elem == [128, 128]
    assert m.layer_sizes[1] == [128, 64, 64, 1]


def test_sizes_and_density():
    for cfg in W.CONFIGS:
        L = W.box_length(cfg.n_atoms)
        assert abs(cfg.n_atoms / L ** 3 - W.water.RHO) < 1e-12
    assert W.CONFIGS[3].n_atoms == 2097153


def test_displacement_stream():
    d1 = W.displacement(1000, 200200255, 1)
    d2 = W.displacement(1000, 200200255, 2)
    assert d1.shape == (1000, 3) and not np.allclose(d1, d2)
    assert 0.008 < d1.std() < 0.012
