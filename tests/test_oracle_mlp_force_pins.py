"""Pins of the oracle's atomic network and forces: special cases, finite differences,
Newton's third law, invariances and an independent PyTorch-autograd derivation
(SURVEY.md 8(c) "What pins each part").  CPU only."""
import math

import numpy as np
import pytest
import torch

import oracle
import workloads as W
from conftest import tiny_model

LN2 = 0.69314718055994531


# ---------------------------------------------------------------- atomic network

def test_mlp_zero_weights():
    sizes = [5, 4, 3, 1]
    nw = 5 * 4 + 4 + 4 * 3 + 3 + 3 + 1
    w = np.zeros(nw)
    w[-4:-1] = [0.5, -1.5, 2.0]     # w3
    w[-1] = 0.25                    # b3
    e, beta = oracle.mlp(sizes, w, np.arange(5.0))
    # hidden activations = softplus(0) = ln 2, sp'(0) = 1/2, beta = 0 because W1 = 0
    assert e == pytest.approx(LN2 * (0.5 - 1.5 + 2.0) + 0.25, rel=1e-15)
    assert np.all(beta == 0.0)


def test_mlp_single_path_by_hand():
    # 1 -> 1 -> 1 -> 1 : E = w3 * sp(w2 * sp(w1 g + b1) + b2) + b3
    w1, b1, w2, b2, w3, b3 = 0.7, -0.2, -1.3, 0.4, 2.5, -0.1
    g = 1.9
    sp = lambda x: math.log1p(math.exp(x))
    sg = lambda x: 1.0 / (1.0 + math.exp(-x))
    z1 = w1 * g + b1
    z2 = w2 * sp(z1) + b2
    e_ref = w3 * sp(z2) + b3
    beta_ref = w3 * sg(z2) * w2 * sg(z1) * w1
    e, beta = oracle.mlp([1, 1, 1, 1], np.array([w1, b1, w2, b2, w3, b3]), np.array([g]))
    assert e == pytest.approx(e_ref, rel=1e-15)
    assert beta[0] == pytest.approx(beta_ref, rel=1e-14)


def test_mlp_softplus_large_arguments():
    # softplus(x) -> x for large x, -> exp(x) for very negative x; no overflow
    e, beta = oracle.mlp([1, 1, 1], np.array([1.0, 0.0, 1.0, 0.0]), np.array([800.0]))
    assert e == 800.0 and beta[0] == pytest.approx(1.0)
    e, beta = oracle.mlp([1, 1, 1], np.array([1.0, 0.0, 1.0, 0.0]), np.array([-800.0]))
    assert e == 0.0 or e < 1e-300


def test_mlp_matches_torch_and_fd():
    model = W.make_model(False)
    sizes = model.layer_sizes[1]
    w = model.weights[1]
    G = np.abs(np.sin(np.arange(sizes[0]) * 1.7)) * 6.0
    e, beta = oracle.mlp(sizes, w, G)
    # library routine: torch linear layers + softplus + autograd
    x = torch.tensor(G, dtype=torch.float64, requires_grad=True)
    h = x
    p = 0
    for l in range(len(sizes) - 1):
        nin, nout = sizes[l], sizes[l + 1]
        Wm = torch.tensor(w[p:p + nin * nout].reshape(nout, nin)); p += nin * nout
        b = torch.tensor(w[p:p + nout]); p += nout
        h = torch.nn.functional.linear(h, Wm, b)
        if l < len(sizes) - 2:
            h = torch.nn.functional.softplus(h)
    h[0].backward()
    assert e == pytest.approx(float(h[0]), rel=1e-13)
    assert np.allclose(beta, x.grad.numpy(), rtol=1e-12, atol=1e-15)
    # finite differences in G
    for s in (0, 7, 51):
        hstep = 1e-5
        Gp, Gm = G.copy(), G.copy()
        Gp[s] += hstep; Gm[s] -= hstep
        fd = (oracle.mlp(sizes, w, Gp, False)[0] - oracle.mlp(sizes, w, Gm, False)[0]) / (2 * hstep)
        assert beta[s] == pytest.approx(fd, rel=1e-7, abs=1e-10)


# ---------------------------------------------------------------- forces

def test_newton_third_law(cfg0):
    sysm, model, om, res = cfg0
    assert np.all(np.abs(res.F.sum(axis=0)) < 1e-9)
    assert np.abs(res.F).max() > 1e-2           # not trivially zero


def _energy_local(om, sysm, pos, atom, rows):
    """E restricted to the centres that can feel `atom` (its neighbours + itself)."""
    sel = np.concatenate([[atom], rows])
    return oracle.centres(om, pos, sysm.types, sysm.box, sel=sel, forces=False, want_g=False).e_total


def test_forces_vs_central_differences(cfg0):
    sysm, model, om, res = cfg0
    off, idx = oracle.neighbor_list(sysm.pos, sysm.box, model.rc + 0.01)   # superset incl. the +-h shell
    w = oracle.wrap(sysm.pos, sysm.box)
    h = 1e-4
    checked = 0
    for atom in (3, 4, 140, 287):
        rows = idx[off[atom]:off[atom + 1]].astype(np.int64)
        # pick atoms whose nearest neighbour is not pathologically close
        d = w[rows] - w[atom]; d -= sysm.box * np.round(d / sysm.box)
        if np.min(np.linalg.norm(d, axis=1)) < 0.5:
            continue
        for x in range(3):
            pp, pm = sysm.pos.copy(), sysm.pos.copy()
            pp[atom, x] += h; pm[atom, x] -= h
            fd = -(_energy_local(om, sysm, pp, atom, rows) - _energy_local(om, sysm, pm, atom, rows)) / (2 * h)
            assert res.F[atom, x] == pytest.approx(fd, rel=1e-6, abs=1e-7)
            checked += 1
    assert checked >= 6


def test_translation_invariance(cfg0):
    sysm, model, om, res = cfg0
    sel = [0, 1, 2, 100, 250]
    for shift in (np.array([0.123456, -7.7, 3.3]), np.array([14.2, -28.4, 0.0])):
        r = oracle.centres(om, sysm.pos + shift, sysm.types, sysm.box, sel=sel, forces=False)
        assert np.allclose(r.e_atom, res.e_atom[sel], rtol=1e-11)
    r = oracle.compute(om, sysm.pos + np.array([0.3, 0.2, -0.9]), sysm.types, sysm.box)
    assert r.e_total == pytest.approx(res.e_total, rel=1e-12)
    assert np.allclose(r.F, res.F, atol=1e-10)


def test_cube_rotation_invariance(cfg0):
    # periodic cube: only the 48 cube symmetries are symmetries (reading C19); take x->y->z->x and a mirror
    sysm, model, om, res = cfg0
    p = sysm.pos[:, [2, 0, 1]].copy()
    p[:, 1] = sysm.box[0] - p[:, 1]
    r = oracle.compute(om, p, sysm.types, sysm.box)
    assert r.e_total == pytest.approx(res.e_total, rel=1e-12)
    Fexp = res.F[:, [2, 0, 1]].copy()
    Fexp[:, 1] *= -1.0
    assert np.allclose(r.F, Fexp, atol=1e-10)
    assert np.allclose(r.e_atom, res.e_atom, rtol=1e-11)


def test_same_element_permutation(cfg0):
    sysm, model, om, res = cfg0
    perm = np.arange(sysm.n_atoms)
    # swap a few H <-> H and O <-> O pairs
    for a, b in ((1, 2), (4, 200), (0, 3), (6, 282)):
        assert sysm.types[a] == sysm.types[b]
        perm[a], perm[b] = perm[b], perm[a]
    r = oracle.compute(om, sysm.pos[perm], sysm.types[perm], sysm.box)
    assert r.e_total == pytest.approx(res.e_total, rel=1e-12)
    assert np.allclose(r.F, res.F[perm], atol=1e-10)


def test_free_rotation_of_isolated_cluster():
    model = W.make_model(False)
    om = oracle.OracleModel(model)
    L = 60.0
    cl = W.make_cluster(24, 5, radius=4.0, L=L)
    r0 = oracle.compute(om, cl.pos, cl.types, cl.box)
    # arbitrary rotation about the box centre
    ax = np.array([0.3, -0.5, 0.81]); ax /= np.linalg.norm(ax)
    th = 1.234
    K = np.array([[0, -ax[2], ax[1]], [ax[2], 0, -ax[0]], [-ax[1], ax[0], 0]])
    R = np.eye(3) + math.sin(th) * K + (1 - math.cos(th)) * K @ K
    p = (cl.pos - L / 2) @ R.T + L / 2
    r1 = oracle.compute(om, p, cl.types, cl.box)
    assert r1.e_total == pytest.approx(r0.e_total, rel=1e-12)
    assert np.allclose(r1.F, r0.F @ R.T, atol=1e-10)
    assert np.all(np.abs(r0.F.sum(0)) < 1e-10)


# ------------------------------------------- independent derivation: dense torch + autograd

def _torch_energy(model, pos, types, box):
    """Dense FP64 evaluation of E(pos) with torch ops; forces by autograd.  Written from the
    definitions (DESIGN.md Readings 1-5), sharing no code with oracle/ or the CUDA library."""
    n = pos.shape[0]
    L = torch.tensor(box)
    d = pos[None, :, :] - pos[:, None, :]          # d[i,j] = r_j - r_i
    d = d - L * torch.round(d / L)
    r2 = (d * d).sum(-1)
    eye = torch.eye(n, dtype=torch.bool)
    r = torch.sqrt(torch.where(eye, torch.ones_like(r2), r2))
    rc = model.rc
    nb = (r2 < rc * rc) & ~eye
    fc = torch.where(nb, 0.5 * (torch.cos(math.pi * r / rc) + 1.0), torch.zeros_like(r))
    t = torch.tensor(types)
    # triplet quantities  [i, j, k]
    cos = (d[:, :, None, :] * d[:, None, :, :]).sum(-1) / (r[:, :, None] * r[:, None, :])
    rjk2 = ((d[:, None, :, :] - d[:, :, None, :]) ** 2).sum(-1)
    rjk = torch.sqrt(torch.where(rjk2 > 0, rjk2, torch.ones_like(rjk2)))
    fjk = torch.where((rjk2 < rc * rc) & (rjk2 > 0), 0.5 * (torch.cos(math.pi * rjk / rc) + 1.0),
                      torch.zeros_like(rjk))
    tri = torch.triu(torch.ones(n, n, dtype=torch.bool), diagonal=1)[None, :, :]
    e_total = 0.0
    for c in range(len(model.elements)):
        rows = model.sf[model.sf["central"] == c]
        cols = []
        for f in rows:
            if f["kind"] == 2:
                g = (torch.exp(-f["eta"] * (r - f["rs"]) ** 2) * fc * (t == int(f["e1"]))[None, :]).sum(1)
            else:
                e1, e2 = int(f["e1"]), int(f["e2"])
                m = ((t[:, None] == e1) & (t[None, :] == e2)) | ((t[:, None] == e2) & (t[None, :] == e1))
                m = (m[None, :, :] & tri).to(pos.dtype)
                X = torch.exp(-f["eta"] * (r2[:, :, None] + r2[:, None, :] + rjk2))
                P = 2.0 ** (1.0 - f["zeta"]) * (1.0 + f["lam"] * cos) ** int(f["zeta"])
                g = (P * X * fc[:, :, None] * fc[:, None, :] * fjk * m).sum((1, 2))
            cols.append(g)
        G = torch.stack(cols, dim=1)
        sizes = model.layer_sizes[c]
        w = model.weights[c]
        h = G
        p = 0
        for l in range(len(sizes) - 1):
            nin, nout = sizes[l], sizes[l + 1]
            Wm = torch.tensor(w[p:p + nin * nout].reshape(nout, nin)); p += nin * nout
            b = torch.tensor(w[p:p + nout]); p += nout
            h = h @ Wm.T + b
            if l < len(sizes) - 2:
                h = torch.nn.functional.softplus(h)
        e_total = e_total + (h[:, 0] * (t == c)).sum()
    return e_total


def test_torch_autograd_cross_check():
    # 60 water-like atoms in a 12.6 A box (> 2 rc) -> ~50 neighbours, fully periodic
    sysm = W.make_water(20, 99, L=12.6)
    model = W.make_model(False)
    om = oracle.OracleModel(model)
    res = oracle.compute(om, sysm.pos, sysm.types, sysm.box)
    pos = torch.tensor(oracle.wrap(sysm.pos, sysm.box), dtype=torch.float64, requires_grad=True)
    e = _torch_energy(model, pos, sysm.types, sysm.box)
    e.backward()
    assert res.e_total == pytest.approx(float(e), rel=1e-12)
    assert np.allclose(res.F, -pos.grad.numpy(), atol=1e-10, rtol=1e-10)


def test_torch_autograd_cross_check_wide_model():
    sysm = W.make_water(12, 5, L=12.2)
    model = W.make_model(True)
    om = oracle.OracleModel(model)
    res = oracle.compute(om, sysm.pos, sysm.types, sysm.box)
    pos = torch.tensor(oracle.wrap(sysm.pos, sysm.box), dtype=torch.float64, requires_grad=True)
    e = _torch_energy(model, pos, sysm.types, sysm.box)
    e.backward()
    assert res.e_total == pytest.approx(float(e), rel=1e-12)
    assert np.allclose(res.F, -pos.grad.numpy(), atol=1e-10, rtol=1e-10)
