"""Pins of the oracle's model-generality features: affine symmetry-function scaling
x = scale (G - shift) in front of the network, and tanh hidden activations.  Pinned to what the
mathematics fixes:
  * shift = 0, scale = 1 changes nothing (bit for bit);
  * a single-path network 1 SF -> 1 neuron -> output evaluated by hand with math.tanh on the
    closed-form two-atom G2 of tests/golden/sf_closed_form.txt;
  * scaling is equivalent to folding it into the first layer (W1' = W1 diag(scale), b1' = b1 - W1 (scale shift)):
    same energies, same forces -> pins the chain rule beta = scale * dE/dx independently of the scaled code path;
  * forces = - central finite differences of the energy with scaling and tanh switched on."""
import copy
import math

import numpy as np
import pytest

import oracle
import workloads as W
from conftest import tiny_model


def _system():
    return W.make_water(24, 5, L=12.5)          # 72 atoms


def _scaled(model, seed=3, activation="softplus"):
    rng = np.random.default_rng(seed)
    m = copy.deepcopy(model)
    m.sf_scaling = [(rng.uniform(0.0, 0.5, n), rng.uniform(0.2, 3.0, n)) for n in m.n_sf_per_elem]
    m.activation = activation
    return m


def test_identity_scaling_changes_nothing():
    sysm = _system()
    model = W.make_model(False)
    r0 = oracle.compute(oracle.OracleModel(model), sysm.pos, sysm.types, sysm.box)
    m1 = copy.deepcopy(model)
    m1.sf_scaling = [(np.zeros(n), np.ones(n)) for n in model.n_sf_per_elem]
    r1 = oracle.compute(oracle.OracleModel(m1), sysm.pos, sysm.types, sysm.box)
    assert np.array_equal(r0.e_atom, r1.e_atom) and np.array_equal(r0.F, r1.F) and np.array_equal(r0.dEdG, r1.dEdG)


def test_single_path_tanh_network_by_hand():
    # two atoms 3 A apart, one radial SF eta = 0.01: G = fc(3) exp(-0.09) = 0.45696559263561409 (golden W1)
    model = tiny_model([(0, 2, 0, 0, 0.01, 0.0, 0.0, 0.0)], hidden=(1,))
    w1, b1, w2, b2 = 0.7, -0.2, 1.3, 0.05
    model.weights = [np.array([w1, b1, w2, b2])]
    model.sf_scaling = [(np.array([0.1]), np.array([2.5]))]
    model.activation = "tanh"
    pos = np.array([[1.0, 1.0, 1.0], [4.0, 1.0, 1.0]])
    r = oracle.compute(oracle.OracleModel(model), pos, np.zeros(2, dtype=np.int32), np.array([20.0, 20.0, 20.0]))
    G = 0.45696559263561409
    t = math.tanh(w1 * 2.5 * (G - 0.1) + b1)
    assert r.e_atom[0] == pytest.approx(w2 * t + b2, rel=1e-14)
    beta = w2 * (1.0 - t * t) * w1 * 2.5
    assert r.dEdG[0, 0] == pytest.approx(beta, rel=1e-13)
    # dG/dr = -0.26668456035269541 (golden W1): force on atom 1 along +x is -2 beta dG/dr (both centres)
    assert r.F[1, 0] == pytest.approx(-2.0 * beta * (-0.26668456035269541), rel=1e-12)
    assert r.F[0, 0] == pytest.approx(-r.F[1, 0], rel=1e-13)


@pytest.mark.parametrize("activation", ["softplus", "tanh"])
def test_scaling_equals_folded_first_layer(activation):
    sysm = _system()
    ms = _scaled(W.make_model(False), activation=activation)
    mf = copy.deepcopy(ms)
    mf.sf_scaling = None
    for e, (shift, scale) in enumerate(ms.sf_scaling):
        n_in, n_h = ms.layer_sizes[e][0], ms.layer_sizes[e][1]
        w = mf.weights[e].copy()
        W1 = w[:n_h * n_in].reshape(n_h, n_in)
        b1 = w[n_h * n_in:n_h * n_in + n_h]
        b1 -= W1 @ (scale * shift)
        W1 *= scale[None, :]
        mf.weights[e] = w
    rs = oracle.compute(oracle.OracleModel(ms), sysm.pos, sysm.types, sysm.box)
    rf = oracle.compute(oracle.OracleModel(mf), sysm.pos, sysm.types, sysm.box)
    assert np.abs(rs.e_atom - rf.e_atom).max() < 1e-12 * np.abs(rf.e_atom).max()
    assert np.abs(rs.F - rf.F).max() < 1e-11
    assert np.abs(rs.dEdG - rf.dEdG).max() < 1e-12 * np.abs(rf.dEdG).max()


def test_forces_vs_central_differences_scaled_tanh():
    sysm = _system()
    om = oracle.OracleModel(_scaled(W.make_model(False), activation="tanh"))
    r = oracle.compute(om, sysm.pos, sysm.types, sysm.box)
    h = 1e-4
    for atom in (0, 7, 40):
        for x in range(3):
            pp, pm = sysm.pos.copy(), sysm.pos.copy()
            pp[atom, x] += h
            pm[atom, x] -= h
            ep = oracle.compute(om, pp, sysm.types, sysm.box, forces=False).e_total
            em = oracle.compute(om, pm, sysm.types, sysm.box, forces=False).e_total
            assert r.F[atom, x] == pytest.approx(-(ep - em) / (2 * h), rel=1e-6, abs=1e-7)
    assert np.abs(r.F.sum(axis=0)).max() < 1e-10
