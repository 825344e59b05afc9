"""Pins of the oracle's per-SF cutoff radii (n2p2 gives every symmetry function its own rc):
an SF with radius rc_s uses fc(r; rc_s) -- zero beyond rc_s -- on the neighbourhood of the global rc.  Pinned
to hand-placed atoms (fc(2; 4) = 1/2, fc(2; 6) = 3/4, fc(3; 6) = 1/2, fc(3; 4) = (1 - 1/sqrt 2)/2), to the model
whose GLOBAL cutoff is that radius (a different neighbour list, the same sum), and to finite differences."""
import math

import numpy as np
import pytest

import oracle
import workloads as W
from conftest import tiny_model

BOX = np.array([40.0, 40.0, 40.0])


def _G(rows, rcs, pos, rc=6.0):
    model = tiny_model(rows, hidden=(2,), rc=rc)
    model.sf_cutoffs = rcs
    r = oracle.compute(oracle.OracleModel(model), np.asarray(pos, dtype=float) + 10.0, np.zeros(len(pos), dtype=np.int32), BOX,
                       forces=False)
    return r.G


def test_radial_hand_values():
    # neighbours at 2 and at 5 of the centre; radial eta = 0.1, rs = 0 and rs = 1
    pos = [[0, 0, 0], [2, 0, 0], [0, -5, 0]]
    rows = [(0, 2, 0, 0, 0.1, 0.0, 0.0, 0.0), (0, 2, 0, 0, 0.1, 0.0, 0.0, 0.0), (0, 2, 0, 0, 0.1, 1.0, 0.0, 0.0)]
    G = _G(rows, [6.0, 4.0, 4.0], pos)
    fc5 = 0.5 * (math.cos(math.pi * 5.0 / 6.0) + 1.0)
    assert G[0, 0] == pytest.approx(math.exp(-0.4) * 0.75 + math.exp(-2.5) * fc5, rel=1e-14)   # rc 6: both
    assert G[0, 1] == pytest.approx(math.exp(-0.4) * 0.5, rel=1e-14)                            # rc 4: the near one, fc = 1/2
    assert G[0, 2] == pytest.approx(math.exp(-0.1) * 0.5, rel=1e-14)
    assert math.exp(-0.4) * 0.5 == pytest.approx(0.33516002301781966, rel=1e-14)


def test_angular_hand_values():
    # right angle at the centre, a = 2, b = 3, c = sqrt 13 = 3.61 (< 4): zeta = 1, lambda = 1 -> 2^0 (1 + 0)
    pos = [[0, 0, 0], [2, 0, 0], [0, 3, 0]]
    rows = [(0, 3, 0, 0, 0.02, 0.0, 1.0, 1.0), (0, 9, 0, 0, 0.02, 0.0, 1.0, 1.0), (0, 3, 0, 0, 0.02, 0.0, 1.0, 1.0)]
    G = _G(rows, [4.0, 4.0, 3.5], pos)
    c = math.sqrt(13.0)
    fc3 = 0.5 * (math.cos(0.75 * math.pi) + 1.0)               # fc(3; 4) = (1 - 1/sqrt 2)/2
    assert fc3 == pytest.approx(0.5 * (1.0 - 1.0 / math.sqrt(2.0)), rel=1e-14)
    fcc = 0.5 * (math.cos(math.pi * c / 4.0) + 1.0)
    assert G[0, 1] == pytest.approx(math.exp(-0.02 * 13.0) * 0.5 * fc3, rel=1e-14)             # wide: fc(2;4) fc(3;4)
    assert G[0, 0] == pytest.approx(math.exp(-0.02 * 26.0) * 0.5 * fc3 * fcc, rel=1e-13)       # narrow: + exp(-eta c^2) fc(c;4)
    assert G[0, 2] == 0.0                                                                       # rc 3.5 < c: no triplet


def test_equal_radii_change_nothing():
    sysm, model = W.build(W.CONFIGS[0])
    r0 = oracle.compute(oracle.OracleModel(model), sysm.pos, sysm.types, sysm.box)
    model.sf_cutoffs = [model.rc] * len(model.sf)
    r1 = oracle.compute(oracle.OracleModel(model), sysm.pos, sysm.types, sysm.box)
    model.sf_cutoffs = None
    assert np.array_equal(r0.G, r1.G) and np.array_equal(r0.F, r1.F) and r0.e_total == r1.e_total


def _mixed_model(rc=6.0):
    rows, rcs = [], []
    for c in range(2):
        for e1 in range(2):
            for rr in (6.0, 4.5, 3.0):
                rows.append((c, 2, e1, 0, 0.08, 0.5, 0.0, 0.0)); rcs.append(rr)
        for (e1, e2) in ((0, 0), (0, 1), (1, 1)):
            rows.append((c, 3, e1, e2, 0.01, 0.0, 1.0, 2.0)); rcs.append(6.0)
            rows.append((c, 3, e1, e2, 0.01, 0.0, -1.0, 1.0)); rcs.append(4.0)
            rows.append((c, 9, e1, e2, 0.02, 0.0, 1.0, 4.0)); rcs.append(5.0)
            rows.append((c, 9, e1, e2, 0.004, 0.0, -1.0, 2.0)); rcs.append(3.2)
    m = tiny_model(rows, n_elem=2, hidden=(5, 4), seed=31, rc=rc)
    m.sf_cutoffs = rcs
    return m


def test_smaller_radius_equals_model_with_that_global_cutoff():
    # the SFs of radius 4.0 / 4.5, evaluated inside the rc = 6 neighbourhood, against a model whose GLOBAL rc is
    # that radius (other neighbour list, no per-SF radii): identical terms, so equal up to summation order
    model = _mixed_model()
    sysm = W.make_water(40, 7, L=13.0)
    G = oracle.compute(oracle.OracleModel(model), sysm.pos, sysm.types, sysm.box, forces=False).G
    for rr in (4.0, 4.5, 3.0, 5.0, 3.2):
        sel = [q for q, r in enumerate(model.sf_cutoffs) if r == rr]
        rows = [tuple(model.sf[q]) for q in sel]
        sub = tiny_model(rows, n_elem=2, hidden=(2,), rc=rr)
        Gs = oracle.compute(oracle.OracleModel(sub), sysm.pos, sysm.types, sysm.box, forces=False).G
        for c in range(2):
            cols_full = [int(np.sum(model.sf["central"][:q] == c)) for q in sel if model.sf["central"][q] == c]
            atoms = np.nonzero(sysm.types == c)[0]
            ref = Gs[atoms][:, :len(cols_full)]
            got = G[atoms][:, cols_full]
            assert np.all(np.abs(got - ref) <= 1e-13 * np.maximum(1.0, np.abs(ref)))
            assert np.abs(ref).max() > 0.0


def test_forces_vs_finite_differences():
    model = _mixed_model()
    sysm = W.make_water(24, 5, L=12.5)
    om = oracle.OracleModel(model)
    r = oracle.compute(om, sysm.pos, sysm.types, sysm.box)
    assert np.abs(r.F.sum(axis=0)).max() < 1e-10
    h = 1e-4
    for atom in (0, 13, 44):
        for x in range(3):
            pp, pm = sysm.pos.copy(), sysm.pos.copy()
            pp[atom, x] += h
            pm[atom, x] -= h
            ep = oracle.compute(om, pp, sysm.types, sysm.box, forces=False).e_total
            em = oracle.compute(om, pm, sysm.types, sysm.box, forces=False).e_total
            assert r.F[atom, x] == pytest.approx(-(ep - em) / (2 * h), rel=1e-6, abs=1e-7)
