"""Pins of the two pieces of oracle glue the full-size parity rests on (CPU only):

  * oracle.forces_on(m): "run the centres N(m) + {m}, read row m" must equal row m of the whole-system
    oracle.compute() -- F, E_i, G_i and the neighbour row: for EVERY atom of configs[0] (2 cells per
    dimension) and of a 12.5 A box with a small two-element table (about 1 ms per centre), and for every 12th
    atom of configs[0] with BASELINE.json's base-52 model.
  * the cell-prefiltered neighbour search (oracle_neighbors_of_cells; used by
    tests/golden/make_fullsize_golden.py for whole-system sums) must return the rows of the brute-force
    scan (the definition) element by element: 1, 2, 3, 4 and 10 cells per dimension, orthorhombic boxes,
    atoms exactly on box faces and outside the box, and -- independently of both -- scipy's periodic k-d tree.
"""
import numpy as np
import pytest
from scipy.spatial import cKDTree

import oracle
import workloads as W


def _all_rows(pos, box, rc, search):
    return oracle.neighbor_rows(pos, box, rc, range(pos.shape[0]), search=search)


def _uniform(box, n, seed):
    from workloads import rng
    k = rng.stream_key(seed, 4711)
    return rng.uniform(k, np.arange(3 * n, dtype=np.uint64)).reshape(n, 3) * np.asarray(box)


def _small_model():
    # 2 elements, radial + narrow angular SFs in every pair group, a real network: the glue under test does not
    # depend on the table, and this one makes EVERY atom affordable (about 1 ms per centre)
    from conftest import tiny_model
    rows = []
    for c in range(2):
        for e1 in range(2):
            rows.append((c, 2, e1, 0, 0.07, 0.3, 0.0, 0.0))
        for (e1, e2) in ((0, 0), (0, 1), (1, 1)):
            rows.append((c, 3, e1, e2, 0.004, 0.0, 1.0 if e1 == e2 else -1.0, 2.0))
    return tiny_model(rows, n_elem=2, hidden=(5, 4), seed=17)


@pytest.mark.parametrize("which", ["config0-every-atom", "box12.5-every-atom", "config0-base52-strided"])
def test_forces_on_equals_rows_of_compute(which, cfg0):
    if which == "config0-base52-strided":
        sysm, model, om, ref = cfg0                     # BASELINE.json's model, every 12th atom
        atoms = np.arange(0, sysm.n_atoms, 12)
    else:
        if which.startswith("config0"):
            sysm = W.build(W.CONFIGS[0])[0]             # 2 cells per dimension
        else:
            sysm = W.make_water(64, 99, L=12.5)         # 192 atoms, L barely above 2 rc
        model = _small_model()
        om = oracle.OracleModel(model)
        ref = oracle.compute(om, sysm.pos, sysm.types, sysm.box)
        atoms = np.arange(sysm.n_atoms)
    got = oracle.forces_on(om, sysm.pos, sysm.types, sysm.box, atoms)
    roff, ridx = oracle.neighbor_list(sysm.pos, sysm.box, model.rc)
    for q, m in enumerate(atoms):
        assert np.array_equal(got.rows[q], ridx[roff[m]:roff[m + 1]])
    # E_i and G_i of the centre itself: the same arithmetic on the same row -> identical
    assert np.array_equal(got.e_atom, ref.e_atom[atoms])
    assert np.array_equal(got.G, ref.G[atoms])
    # F_m: the same terms summed in another order (row m of N(m)+{m} vs all centres) -> rounding only
    scale = np.abs(ref.F).max()
    assert np.abs(got.F - ref.F[atoms]).max() <= 1e-13 * max(1.0, scale)
    # and a wrong glue (forgetting the centre's own term, or a neighbour's) would be far off
    assert scale > 1e-3


@pytest.mark.parametrize("box,n,seed", [
    ((14.2, 14.2, 14.2), 288, 1),           # 2 x 2 x 2 cells
    ((12.6, 18.7, 31.0), 600, 2),           # 2 x 3 x 5
    ((12.0, 12.0, 12.0), 200, 3),           # exactly 2 rc: nc = 1 (12 / (6 (1 + 1e-9)) < 2)
    ((24.5, 13.0, 36.1), 700, 4),           # 4 x 2 x 6
    ((61.0, 60.5, 62.5), 3000, 5),          # 10 cells per dimension, sparse
])
def test_cell_search_equals_brute_force(box, n, seed):
    box = np.array(box)
    pos = _uniform(box, n, seed)
    # atoms exactly on faces / corners, and copies far outside the box (wrapped by the oracle)
    pos[0] = (0.0, 0.0, 0.0)
    pos[1] = (box[0], 0.5 * box[1], box[2])
    pos[2] = (np.nextafter(box[0], 0.0), 0.0, np.nextafter(box[2], 0.0))
    pos[3] = (-1e-17, -1e-300, 3.0)                      # wraps to exactly L in x (rounding) and in y
    pos[4:20] += 3.0 * box
    pos[20:40] -= 2.0 * box
    a = _all_rows(pos, box, 6.0, "brute")
    b = _all_rows(pos, box, 6.0, "cells")
    assert sum(len(r) for r in a) > 0
    for ra, rb in zip(a, b):
        assert np.array_equal(ra, rb)
    # independent library search on the wrapped positions (pairs whose distance is within 1e-9 of rc excluded)
    w = oracle.wrap(pos, box)
    w = np.where(w >= box, 0.0, w)                       # scipy wants [0, L)
    tree = cKDTree(w, boxsize=box)
    inner = tree.query_ball_point(w, 6.0 - 1e-9)
    outer = tree.query_ball_point(w, 6.0 + 1e-9)
    for m in range(n):
        row = set(b[m].tolist())
        assert set(inner[m]) - {m} <= row <= set(outer[m]) - {m}


def test_cell_search_whole_pipeline_identical():
    # oracle.centres(search="cells") = oracle.centres(search="brute"), every output bit for bit
    sysm, model = W.build(W.CONFIGS[0])
    om = oracle.OracleModel(model)
    a = oracle.centres(om, sysm.pos, sysm.types, sysm.box, None, rows=True)
    b = oracle.centres(om, sysm.pos, sysm.types, sysm.box, None, rows=True, search="cells")
    for k in ("e_atom", "G", "dEdG", "nbr_count", "F", "row_off", "row_idx"):
        assert np.array_equal(getattr(a, k), getattr(b, k)), k
    roff, ridx = oracle.neighbor_list(sysm.pos, sysm.box, model.rc)
    assert np.array_equal(a.row_off, roff) and np.array_equal(a.row_idx, ridx)


def test_cell_search_sampled_rows_of_config1():
    # 10 cells per dimension at the workload's density; rows of boundary-cell atoms and of a random sample
    sysm, model = W.build(W.CONFIGS[1])
    L = sysm.box[0]
    x = sysm.pos
    picks = [int(np.argmin(x[:, c])) for c in range(3)] + [int(np.argmax(x[:, c])) for c in range(3)]
    picks += list(np.random.RandomState(5).choice(sysm.n_atoms, 150, replace=False))
    a = oracle.neighbor_rows(sysm.pos, sysm.box, model.rc, picks, "brute")
    b = oracle.neighbor_rows(sysm.pos, sysm.box, model.rc, picks, "cells")
    for ra, rb in zip(a, b):
        assert np.array_equal(ra, rb)
    assert 80 < np.mean([len(r) for r in a]) < 100 and L > 60
