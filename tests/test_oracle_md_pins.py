"""Pins of the MD oracle (oracle/md.py, velocity Verlet around the oracle forces): things the
mathematics fixes, none of them computed by the code under test.
  * the acceleration unit from the CODATA-2018 values of e and the atomic mass constant, and the
    header's NNP_ACC_UNIT equal to it;
  * time reversibility of velocity Verlet (forward n steps, flip velocities, n steps: back at the start);
  * second-order accuracy: halving dt divides the energy error at a fixed time by ~4;
  * total momentum conserved (the forces sum to zero), kinetic energy of a hand-made state."""
import os
import re

import numpy as np

import oracle
import workloads as W
from oracle import md

MASS = (1.008, 15.999)      # H, O in amu (element order of the models)


def _small():
    sysm = W.make_water(24, 77, L=12.5)          # 72 atoms, L > 2 rc
    model = W.make_model(False)
    rng = np.random.default_rng(5)
    vel = rng.normal(0.0, 0.005, size=(sysm.n_atoms, 3))   # A/fs, ~ thermal
    m = np.asarray(MASS)[sysm.types][:, None]
    vel -= (m * vel).sum(axis=0) / m.sum()
    return sysm, oracle.OracleModel(model), vel


def test_acceleration_unit_and_header_constant():
    assert md.ACC_UNIT == (1.602176634e-19 / 1e-10) / 1.66053906660e-27 * 1e10 / 1e30
    assert abs(md.ACC_UNIT - 9.6485332157e-3) < 1e-12
    hdr = open(os.path.join(os.path.dirname(__file__), "..", "include", "nnp.h")).read()
    val = float(re.search(r"#define NNP_ACC_UNIT\s+([0-9.eE+-]+)", hdr).group(1))
    assert val == md.ACC_UNIT


def test_kinetic_energy_by_hand():
    # one O atom at 0.01 A/fs: m v^2 / 2 = 15.999 * 1e-4 / 2 amu A^2/fs^2 = 7.9995e-4 / ACC_UNIT eV
    e = md.kinetic_energy(np.array([[0.01, 0.0, 0.0]]), np.array([1]), MASS)
    assert abs(e - 7.9995e-4 / md.ACC_UNIT) < 1e-15 * e
    assert abs(e - 0.0829089) < 1e-6          # eV, worked by hand: 7.9995e-4 / 9.6485332e-3


def test_time_reversibility():
    sysm, om, vel = _small()
    x1, v1, _, _, _ = md.run(om, sysm.pos, vel, sysm.types, sysm.box, MASS, 0.5, 6)
    x2, v2, _, _, _ = md.run(om, x1, -v1, sysm.types, sysm.box, MASS, 0.5, 6)
    assert np.abs(x2 - sysm.pos).max() < 1e-11
    assert np.abs(v2 + vel).max() < 1e-12


def test_second_order_energy_error_and_momentum():
    sysm, om, vel = _small()
    errs = []
    for dt, n in ((1.0, 8), (0.5, 16)):
        x, v, F, ep, ek = md.run(om, sysm.pos, vel, sysm.types, sysm.box, MASS, dt, n)
        e = np.array(ep) + np.array(ek)
        errs.append(np.abs(e - e[0]).max())
        m = np.asarray(MASS)[sysm.types][:, None]
        assert np.abs((m * v).sum(axis=0)).max() < 1e-10          # momentum stays zero
    assert errs[0] > 0 and 2.5 < errs[0] / errs[1] < 6.0           # O(dt^2)
    assert errs[1] < 1e-3 * abs(ep[0])
