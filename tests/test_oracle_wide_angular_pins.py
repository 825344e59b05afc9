"""Pins of the oracle's WIDE angular symmetry function (kind 9 in n2p2's numbering):
    G = 2^(1-zeta) sum_{j<k} (1 + lambda cos)^zeta exp(-eta (a^2 + b^2)) fc(a) fc(b)
-- no r_jk in the exponent and no r_jk cutoff.  Pinned to hand-placed three-atom configurations (rc = 6, so
fc(3) = 1/2, fc(2) = 3/4 exactly), to the narrow function where the two must agree or differ in a known way,
and to finite differences / Newton's third law for the forces."""
import math

import numpy as np
import pytest

import oracle
import workloads as W
from conftest import tiny_model

BOX = np.array([40.0, 40.0, 40.0])


def _G(rows, pos):
    model = tiny_model(rows, hidden=(2,))
    r = oracle.compute(oracle.OracleModel(model), np.asarray(pos, dtype=float) + 10.0, np.zeros(len(pos), dtype=np.int32), BOX,
                       forces=False)
    return r.G


def test_equilateral_triangle_side_3():
    # centre at a vertex: a = b = 3, cos = 1/2, fc fc = 1/4, exp(-eta 18); zeta = 1: (1 + lambda/2)
    pos = [[0, 0, 0], [3, 0, 0], [1.5, 1.5 * math.sqrt(3.0), 0]]
    G = _G([(0, 9, 0, 0, 0.01, 0.0, 1.0, 1.0), (0, 9, 0, 0, 0.01, 0.0, -1.0, 1.0), (0, 9, 0, 0, 0.01, 0.0, 1.0, 2.0)], pos)
    x = math.exp(-0.18) * 0.25                      # 0.20881755285281800
    assert G[0, 0] == pytest.approx(1.5 * x, rel=1e-14)            # 0.31322632927922700
    assert G[0, 1] == pytest.approx(0.5 * x, rel=1e-14)
    assert G[0, 2] == pytest.approx(0.5 * 2.25 * x, rel=1e-14)     # 2^(1-2) (3/2)^2
    assert 1.5 * x == pytest.approx(0.313226329279227, rel=1e-13)


def test_far_pair_counts_in_wide_not_in_narrow():
    # j, k at +-3.5 on a line through the centre: r_jk = 7 > rc -> narrow G3 = 0, wide G9 = 2 (1 - lambda)^... with cos = -1
    pos = [[0, 0, 0], [3.5, 0, 0], [-3.5, 0, 0]]
    G = _G([(0, 3, 0, 0, 0.01, 0.0, -1.0, 1.0), (0, 9, 0, 0, 0.01, 0.0, -1.0, 1.0), (0, 9, 0, 0, 0.01, 0.0, 1.0, 4.0)], pos)
    fc35 = 0.5 * (math.cos(math.pi * 3.5 / 6.0) + 1.0)
    assert G[0, 0] == 0.0
    assert G[0, 1] == pytest.approx(2.0 * math.exp(-0.01 * 24.5) * fc35 * fc35, rel=1e-14)
    assert G[0, 2] == 0.0                           # (1 + cos)^4 = 0


def test_wide_equals_narrow_times_known_factor():
    # one triangle with r_jk < rc: narrow = wide * exp(-eta c^2) * fc(c)
    pos = [[0, 0, 0], [2, 0, 0], [0, 3, 0]]
    G = _G([(0, 3, 0, 0, 0.02, 0.0, 1.0, 2.0), (0, 9, 0, 0, 0.02, 0.0, 1.0, 2.0)], pos)
    c = math.sqrt(13.0)
    assert G[0, 0] == pytest.approx(G[0, 1] * math.exp(-0.02 * 13.0) * 0.5 * (math.cos(math.pi * c / 6.0) + 1.0), rel=1e-13)
    # right angle at the centre: (1 + 0)^2 / 2, a = 2, b = 3
    assert G[0, 1] == pytest.approx(0.5 * math.exp(-0.02 * 13.0) * 0.75 * 0.5, rel=1e-14)


def _wide_model():
    rows = []
    for c in range(2):
        for e1 in range(2):
            rows.append((c, 2, e1, 0, 0.05, 0.0, 0.0, 0.0))
        for (e1, e2) in ((0, 0), (0, 1), (1, 1)):
            rows.append((c, 9, e1, e2, 0.004, 0.0, 1.0, 2.0))
            rows.append((c, 9, e1, e2, 0.010, 0.0, -1.0, 1.0))
            rows.append((c, 3, e1, e2, 0.004, 0.0, 1.0, 4.0))      # mixed with a narrow one in the same group
    return tiny_model(rows, n_elem=2, hidden=(5, 4), seed=21)


def test_forces_vs_finite_differences_and_newton():
    model = _wide_model()
    sysm = W.make_water(24, 5, L=12.5)
    om = oracle.OracleModel(model)
    r = oracle.compute(om, sysm.pos, sysm.types, sysm.box)
    assert np.abs(r.F.sum(axis=0)).max() < 1e-10
    h = 1e-4
    for atom in (1, 20, 50):
        for x in range(3):
            pp, pm = sysm.pos.copy(), sysm.pos.copy()
            pp[atom, x] += h
            pm[atom, x] -= h
            ep = oracle.compute(om, pp, sysm.types, sysm.box, forces=False).e_total
            em = oracle.compute(om, pm, sysm.types, sysm.box, forces=False).e_total
            assert r.F[atom, x] == pytest.approx(-(ep - em) / (2 * h), rel=1e-6, abs=1e-7)
    # translation by an arbitrary vector and same-element permutation leave the energy alone
    r2 = oracle.compute(om, sysm.pos + np.array([0.3, -1.1, 2.2]), sysm.types, sysm.box, forces=False)
    assert r2.e_total == pytest.approx(r.e_total, rel=1e-12)
