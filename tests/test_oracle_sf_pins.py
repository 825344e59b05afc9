"""Pins of the oracle's geometry, cutoff and symmetry functions against closed forms,
a library neighbour search and identities (SURVEY.md 8(c) "What pins each part").
CPU only."""
import math
import os

import numpy as np
import pytest
from scipy.spatial import cKDTree

import oracle
import workloads as W
from conftest import tiny_model

GOLD = os.path.join(os.path.dirname(__file__), "golden", "sf_closed_form.txt")
BOX = np.array([40.0, 40.0, 40.0])
C0 = np.array([20.0, 20.0, 20.0])


def _rows():
    out = []
    for line in open(GOLD):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        t = line.split()
        out.append((t[0], int(t[1]), float(t[2]), float(t[3]), float(t[4]), float(t[5]),
                    float(t[6]), float(t[7])))
    return out


def _geometry(case, d):
    """positions with the CENTRE as atom 0"""
    if case == "pair":
        return np.array([[0, 0, 0], [d, 0, 0]], dtype=float)
    if case == "equi":
        return np.array([[0, 0, 0], [3, 0, 0], [1.5, 1.5 * math.sqrt(3.0), 0]], dtype=float)
    if case == "rightc":
        return np.array([[0, 0, 0], [3, 0, 0], [0, 3, 0]], dtype=float)
    if case == "rightb":          # centre at a base corner of the same triangle
        return np.array([[3, 0, 0], [0, 0, 0], [0, 3, 0]], dtype=float)
    if case == "colli":
        return np.array([[0, 0, 0], [2, 0, 0], [-2, 0, 0]], dtype=float)
    if case == "far":
        return np.array([[0, 0, 0], [3.5, 0, 0], [-3.5, 0, 0]], dtype=float)
    raise KeyError(case)


def _G_centre0(pos, kind, eta, lam, zeta, rs=0.0):
    m = tiny_model([(0, kind, 0, 0, eta, rs, lam, zeta)])
    om = oracle.OracleModel(m)
    types = np.zeros(len(pos), dtype=np.int32)
    # rotate the geometry out of the axes so no component is special, then shift
    th = 0.7
    R = np.array([[math.cos(th), -math.sin(th), 0], [math.sin(th), math.cos(th), 0], [0, 0, 1.0]])
    R2 = np.array([[1, 0, 0], [0, math.cos(0.4), -math.sin(0.4)], [0, math.sin(0.4), math.cos(0.4)]])
    p = pos @ (R @ R2).T + C0
    r = oracle.centres(om, p, types, BOX, sel=[0], forces=False)
    return r.G[0, 0], r.nbr_count[0]


@pytest.mark.parametrize("row", _rows(), ids=lambda r: "%s-k%d-d%g-eta%g-l%g-z%g" % r[:6])
def test_closed_form(row):
    case, kind, d, eta, lam, zeta, g_exp, dg_exp = row
    if case == "fc":
        assert oracle.fc(d, 6.0) == pytest.approx(g_exp, rel=2e-15, abs=1e-16)
        return
    g, nn = _G_centre0(_geometry(case, d), kind, eta, lam, zeta)
    if g_exp == 0.0:
        assert abs(g) < 1e-15      # cos = -1 up to rounding of the rotated geometry
    else:
        assert g == pytest.approx(g_exp, rel=5e-14)
    if case == "far":
        assert nn == 2            # both ARE neighbours of the centre; only r_jk > rc kills it
    if not math.isnan(dg_exp):
        # dG/dr from the oracle's FORCE output: one SF, identity network E = G  =>  F_j = -dG/dr * u/r
        m = tiny_model([(0, kind, 0, 0, eta, 0.0, lam, zeta)], hidden=())
        m.layer_sizes = [[1, 1]]
        m.weights = [np.array([1.0, 0.0])]
        om = oracle.OracleModel(m)
        p = _geometry(case, d) + C0
        r = oracle.centres(om, p, np.zeros(2, dtype=np.int32), BOX, sel=[0])
        # centre 0 only: force on atom 1 is -dG/dr along +x
        assert r.F[1, 0] == pytest.approx(-dg_exp, rel=5e-14)
        assert r.F[0, 0] == pytest.approx(dg_exp, rel=5e-14)
        assert abs(r.F[1, 1]) < 1e-18 and abs(r.F[1, 2]) < 1e-18


def test_fc_edges():
    assert oracle.fc(6.0, 6.0) == 0.0 and oracle.fc(7.0, 6.0) == 0.0
    assert oracle.fc(0.0, 6.0) == 1.0
    assert oracle.dfc(6.5, 6.0) == 0.0
    # fc' by central differences
    for r in (0.5, 2.2, 5.9):
        h = 1e-6
        fd = (oracle.fc(r + h, 6.0) - oracle.fc(r - h, 6.0)) / (2 * h)
        assert oracle.dfc(r, 6.0) == pytest.approx(fd, rel=1e-8)


def test_rs_shift_closed_form():
    # radial with Rs: G = fc(d) exp(-eta (d-Rs)^2); d = 2, Rs = 1.5, eta = 0.5 -> 0.75 exp(-0.125)
    g, _ = _G_centre0(_geometry("pair", 2.0), 2, 0.5, 0, 0, rs=1.5)
    assert g == pytest.approx(0.75 * math.exp(-0.125), rel=1e-14)


def test_min_image_through_boundary():
    # W7: atoms at x = 0.5 and L - 0.5 are 1.0 apart through the boundary
    L = 14.2
    m = tiny_model([(0, 2, 0, 0, 0.01, 0.0, 0, 0)])
    om = oracle.OracleModel(m)
    p = np.array([[0.5, 3.0, 3.0], [L - 0.5, 3.0, 3.0]])
    r = oracle.centres(om, p, np.zeros(2, dtype=np.int32), np.array([L, L, L]), forces=False)
    fc1 = (2.0 + math.sqrt(3.0)) / 4.0
    assert r.G[0, 0] == pytest.approx(fc1 * math.exp(-0.01), rel=1e-13)
    assert r.G[1, 0] == pytest.approx(fc1 * math.exp(-0.01), rel=1e-13)
    # and unwrapped input (outside the box by whole periods) gives the same answer
    p2 = p + np.array([[2 * L, -L, 0.0], [-3 * L, L, L]])
    r2 = oracle.centres(om, p2, np.zeros(2, dtype=np.int32), np.array([L, L, L]), forces=False)
    assert r2.G[0, 0] == pytest.approx(r.G[0, 0], rel=1e-12)


def test_wrap_definition():
    box = np.array([10.0, 7.0, 3.0])
    p = np.array([[-0.25, 7.0, 2.999], [23.5, -13.0, -1e-18], [10.0, 0.0, 3.0]])
    w = oracle.wrap(p, box)
    assert np.allclose(w[0], [9.75, 0.0, 2.999])
    assert np.allclose(w[1], [3.5, 1.0, 3.0])       # -1e-18 + 3 rounds to 3.0 (documented: may equal L)
    assert np.allclose(w[2], [0.0, 0.0, 0.0])


def test_element_pair_indexing_water_molecule():
    # W6: one O + 2 H.  Central O sees only the {H,H} pair group; central H only {H,O}.
    model = W.make_model(False)
    om = oracle.OracleModel(model)
    pos = np.array([[20, 20, 20], [20.96, 20, 20], [19.76, 20.93, 20]], dtype=float)
    types = np.array([W.TYPE_O, W.TYPE_H, W.TYPE_H], dtype=np.int32)
    r = oracle.centres(om, pos, types, BOX, forces=False)
    sf = model.sf
    for atom, tc in enumerate(types):
        rows = sf[sf["central"] == tc]
        for s, f in enumerate(rows):
            g = r.G[atom, s]
            if f["kind"] == 2:
                # O centre: H neighbours only; H centre: one H and one O neighbour
                expect_nonzero = (f["e1"] == W.TYPE_H) if tc == W.TYPE_O else True
            else:
                pair = (int(f["e1"]), int(f["e2"]))
                expect_nonzero = (pair == (0, 0)) if tc == W.TYPE_O else (pair == (0, 1))
            if f["kind"] == 3 and f["lam"] == 1.0 and expect_nonzero:
                assert g > 0
            if not expect_nonzero:
                assert g == 0.0, (atom, s, f)
    assert np.count_nonzero(r.G[0]) > 8


def test_neighbours_vs_kdtree(cfg0):
    sysm, model, om, res = cfg0
    off, idx = oracle.neighbor_list(sysm.pos, sysm.box, model.rc)
    tree = cKDTree(oracle.wrap(sysm.pos, sysm.box) % sysm.box[0], boxsize=sysm.box[0])
    rows = tree.query_ball_point(tree.data, r=model.rc)
    n = sysm.n_atoms
    total = 0
    for i in range(n):
        mine = idx[off[i]:off[i + 1]]
        ref = sorted(j for j in rows[i] if j != i)
        assert list(mine) == ref
        total += len(ref)
    assert total == off[-1]
    assert np.array_equal(res.nbr_count, np.diff(off))
    # symmetry j in N(i) <=> i in N(j)
    pairs = set()
    for i in range(n):
        for j in idx[off[i]:off[i + 1]]:
            pairs.add((i, int(j)))
    assert all((j, i) in pairs for (i, j) in pairs)
    # ideal-gas expectation rho * 4/3 pi rc^3 = 91.0 (statistical sanity)
    assert 85 < total / n < 97


def test_tiny_box_two_cells_brute_force():
    # box just over 2 rc: every atom pair has ONE minimum image; compare with explicit image loop
    L = 12.5
    rc = 6.0
    key_sys = W.make_water(20, 11, L=L)
    pos = key_sys.pos
    off, idx = oracle.neighbor_list(pos, key_sys.box, rc)
    n = pos.shape[0]
    for i in range(n):
        ref = []
        for j in range(n):
            if j == i:
                continue
            best = min(np.sum((pos[j] - pos[i] + np.array([a, b, c]) * L) ** 2)
                       for a in (-1, 0, 1) for b in (-1, 0, 1) for c in (-1, 0, 1))
            if best < rc * rc:
                ref.append(j)
        assert list(idx[off[i]:off[i + 1]]) == ref


def test_angular_identities(cfg0):
    sysm, model, om, res = cfg0
    sf = model.sf
    # G3(lambda=+1, zeta=1) + G3(lambda=-1, zeta=1) = 2 sum X C  (angle-free); compare with a direct
    # numpy evaluation of sum_{j<k} X C over the oracle's own neighbour rows for a few atoms
    off, idx = oracle.neighbor_list(sysm.pos, sysm.box, model.rc)
    w = oracle.wrap(sysm.pos, sysm.box)
    L = sysm.box[0]
    for atom in (0, 1, 17, 100):
        tc = sysm.types[atom]
        rows = sf[sf["central"] == tc]
        nb = idx[off[atom]:off[atom + 1]]
        u = w[nb] - w[atom]
        u -= L * np.round(u / L)
        a = np.linalg.norm(u, axis=1)
        fca = 0.5 * (np.cos(np.pi * a / 6.0) + 1.0)
        for (e1, e2) in ((0, 0), (0, 1), (1, 1)):
            sp = [s for s, f in enumerate(rows) if f["kind"] == 3 and f["e1"] == e1 and f["e2"] == e2
                  and f["eta"] == 0.001 and f["zeta"] == 1.0]
            assert len(sp) == 2
            tot = 0.0
            tn = sysm.types[nb]
            for j in range(len(nb)):
                for k in range(j + 1, len(nb)):
                    if sorted((tn[j], tn[k])) != [e1, e2]:
                        continue
                    c = np.linalg.norm(u[k] - u[j])
                    if c >= 6.0:
                        continue
                    tot += (math.exp(-0.001 * (a[j] ** 2 + a[k] ** 2 + c * c)) * fca[j] * fca[k]
                            * 0.5 * (math.cos(math.pi * c / 6.0) + 1.0))
            assert res.G[atom, sp[0]] + res.G[atom, sp[1]] == pytest.approx(2.0 * tot, rel=1e-11)


def test_mirror_image_leaves_G_unchanged(cfg0):
    sysm, model, om, res = cfg0
    p = sysm.pos.copy()
    p[:, 0] = sysm.box[0] - p[:, 0]
    sel = [0, 5, 77, 200]
    r = oracle.centres(om, p, sysm.types, sysm.box, sel=sel, forces=False)
    assert np.allclose(r.G, res.G[sel], rtol=1e-11, atol=1e-13)
