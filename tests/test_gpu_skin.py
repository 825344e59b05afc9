"""Neighbour-list reuse with a Verlet skin (nnp_set_neighbor_skin, PAPER.md L48 / L116): whatever a call
decides -- rebuild or filter the candidate list of an earlier call -- its results are those of a fresh build: neighbour
sets bit-exact, energy and forces within BASELINE.json's tolerances of the oracle, which knows nothing about skins."""
import numpy as np
import pytest
import torch

import oracle
import workloads as W
from conftest import tiny_model

pytestmark = pytest.mark.gpu
MASS = (1.008, 15.999)


def _call(nnp, pos, types, box):
    dev = torch.device("cuda", 0)
    p = torch.tensor(np.ascontiguousarray(pos), dtype=torch.float64, device=dev)
    t = torch.tensor(np.ascontiguousarray(types), dtype=torch.int32, device=dev)
    e_atom, e_total, force = nnp.compute(p, t, box)
    torch.cuda.synchronize()
    return e_atom.cpu().numpy(), float(e_total.item()), force.cpu().numpy()


def _against_oracle(nnp, om, rc, pos, types, box):
    e_atom, e_total, force = _call(nnp, pos, types, box)
    n = len(types)
    off, idx = nnp.neighbors(n)
    roff, ridx = oracle.neighbor_list(pos, box, rc)
    assert np.array_equal(off.cpu().numpy(), roff)
    assert np.array_equal(idx.cpu().numpy(), ridx)
    ref = oracle.compute(om, pos, types, box)
    assert abs(e_total - ref.e_total) <= 1e-10 * abs(ref.e_total)
    assert np.all(np.abs(e_atom - ref.e_atom) <= 1e-10 * np.abs(ref.e_atom).max())
    assert np.abs(force - ref.F).max() <= 1e-8


def test_skin_sequence_water():
    from paper_2002_00054_b200 import NNP
    sysm = W.make_water(150, 5, L=16.7)                   # 450 atoms, 2 cells of rc + skin per dimension
    model = W.make_model(False)
    om = oracle.OracleModel(model)
    nnp = NNP.from_model(model)
    plain_bytes = nnp.workspace_bytes(sysm.n_atoms)
    nnp.set_neighbor_skin(0.6)
    assert nnp.workspace_bytes(sysm.n_atoms) > plain_bytes
    rs = np.random.RandomState(11)
    pos = sysm.pos.copy()
    expect = []                                           # rebuild expected at call k?
    seq = []
    seq.append(pos.copy()); expect.append(True)           # first call on this workspace
    step = rs.uniform(-0.05, 0.05, size=pos.shape)        # |d| <= 0.087 per call
    for k in range(3):                                    # cumulative |d| <= 0.26 < skin/2
        pos = pos + step
        seq.append(pos.copy()); expect.append(False)
    pos = pos + step                                      # 4 steps: the largest displacement is now ~0.33 > 0.3
    assert np.linalg.norm(4 * step, axis=1).max() > 0.3
    seq.append(pos.copy()); expect.append(True)
    pos = pos + np.array([sysm.box[0], -2 * sysm.box[1], 0.0])     # whole box vectors: the same wrapped positions
    seq.append(pos.copy()); expect.append(False)
    for k in range(5):                                    # drift through the periodic boundary, 0.05 per call
        pos = pos + np.array([0.05, 0.0, 0.0])
        seq.append(pos.copy()); expect.append(False)
    pos = pos + np.array([0.06, 0.0, 0.0])                # 0.31 since the rebuild
    seq.append(pos.copy()); expect.append(True)
    pos = pos.copy(); pos[17] += np.array([0.0, 1.3, -0.8])        # ONE atom jumps
    seq.append(pos.copy()); expect.append(True)
    seq.append(pos.copy()); expect.append(False)          # nothing moved
    crossed = np.any(np.floor(seq[5] / sysm.box) != np.floor(seq[10] / sysm.box))
    assert crossed                                        # some atom did leave the box on the way
    rebuilds = 0
    for k, (p, e) in enumerate(zip(seq, expect)):
        _against_oracle(nnp, om, model.rc, p, sysm.types, sysm.box)
        calls, rb = nnp.neighbor_rebuilds()
        assert calls == k + 1
        assert (rb - rebuilds == 1) == e, "call %d: rebuild expected %s" % (k, e)
        rebuilds = rb
    # a type change alone forces a rebuild (the sorted order is by element)
    types = sysm.types.copy()
    o, h = np.nonzero(types == W.TYPE_O)[0][3], np.nonzero(types == W.TYPE_H)[0][8]
    types[o], types[h] = W.TYPE_H, W.TYPE_O
    _against_oracle(nnp, om, model.rc, seq[-1], types, sysm.box)
    assert nnp.neighbor_rebuilds()[1] == rebuilds + 1
    # another box: host-side check
    box2 = sysm.box * 1.01
    _against_oracle(nnp, om, model.rc, seq[-1], types, box2)
    assert nnp.neighbor_rebuilds()[1] == rebuilds + 2
    # invalidate
    nnp.invalidate_neighbors()
    _against_oracle(nnp, om, model.rc, seq[-1], types, box2)
    assert nnp.neighbor_rebuilds()[1] == rebuilds + 3
    # back to no skin: counters reset, every call searches the cells
    nnp.set_neighbor_skin(0.0)
    assert nnp.workspace_bytes(sysm.n_atoms) == plain_bytes
    _against_oracle(nnp, om, model.rc, seq[3], sysm.types, sysm.box)
    assert nnp.neighbor_rebuilds() == (0, 0)
    nnp.close()


def test_skin_sequence_metal_small_rows():
    # fcc Ni-like cell, max_neighbors = 32: the 8-lanes-per-atom filter and the small-neighbourhood kernels
    from paper_2002_00054_b200 import NNP
    sysm, model = W.build(W.Config("fcc6", 6, False, 1, 11, 12, None, "metal"))
    om = oracle.OracleModel(model)
    nnp = NNP.from_model(model)
    nnp.set_max_neighbors(32)
    nnp.set_neighbor_skin(0.4)
    rs = np.random.RandomState(5)
    pos = sysm.pos.copy()
    rb_before = 0
    pattern = []
    for k in range(7):
        _against_oracle(nnp, om, model.rc, pos, sysm.types, sysm.box)
        rb = nnp.neighbor_rebuilds()[1]
        pattern.append(rb - rb_before)
        rb_before = rb
        pos = pos + rs.uniform(-0.04, 0.04, size=pos.shape)
    assert pattern[0] == 1 and 1 <= sum(pattern) < 7      # the random walk needs a rebuild now and then, not every call
    nnp.close()


def test_skin_errors_and_limits():
    from paper_2002_00054_b200 import NNP, NNPError
    sysm, model = W.build(W.CONFIGS[0])                   # L = 14.2
    nnp = NNP.from_model(model)
    for bad in (-0.1, float("nan"), model.rc + 1.0):
        with pytest.raises(NNPError):
            nnp.set_neighbor_skin(bad)
    nnp.set_neighbor_skin(1.2)                            # 2 (rc + skin) = 14.4 > L
    with pytest.raises(NNPError) as ei:
        _call(nnp, sysm.pos, sysm.types, sysm.box)
    assert "BOX" in str(ei.value).upper()
    nnp.close()


def test_md_run_with_skin_matches_md_run_without():
    # the CUDA-graph replay of nnp_md_run takes the rebuild decision on the device: same trajectory, fewer rebuilds
    from paper_2002_00054_b200 import NNP
    sysm = W.make_water(700, 4242)
    model = W.make_model(False)
    rng = np.random.default_rng(9)
    vel = rng.normal(0.0, 0.005, size=(sysm.n_atoms, 3))
    dev = torch.device("cuda", 0)
    out = []
    for skin in (0.0, 0.5):
        nnp = NNP.from_model(model)
        nnp.set_neighbor_skin(skin)
        pos_d = torch.tensor(sysm.pos, dtype=torch.float64, device=dev)
        vel_d = torch.tensor(vel, dtype=torch.float64, device=dev)
        typ_d = torch.tensor(sysm.types, dtype=torch.int32, device=dev)
        state = nnp.compute(pos_d, typ_d, sysm.box)
        nnp.md_run(120, 0.05, MASS, pos_d, vel_d, typ_d, sysm.box, state)
        nnp.sync_status()
        out.append((pos_d.cpu().numpy(), state[2].cpu().numpy(), float(state[1].item()), nnp.neighbor_rebuilds()))
        nnp.close()
    (x0, f0, e0, s0), (x1, f1, e1, s1) = out
    assert s0 == (0, 0)
    # 120 steps + the first call; the synthetic model's forces reach 20 eV/A, so the fastest H atom covers skin/2 in ~20 steps
    assert s1[0] == 121 and 2 <= s1[1] <= 60, s1
    assert np.abs(x1 - x0).max() < 1e-8                   # summation order differs (row order), nothing else
    assert np.abs(f1 - f0).max() < 1e-8
    assert abs(e1 - e0) < 1e-10 * abs(e0)
