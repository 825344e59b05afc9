"""Parity of the CUDA path (through the C ABI) against the CPU oracle, element by element, on the
same seeded inputs.  Tolerances (BASELINE.json north_star):
  neighbour sets bit-exact (sorted index lists); total energy relative 1e-10;
  force components absolute 1e-8 eV/A; e_atom abs 1e-10*max|E_i|; G abs 1e-11*max(1,|G|)."""
import json
import math
import os

import numpy as np
import pytest
import torch

import oracle
import workloads as W
from conftest import tiny_model

pytestmark = pytest.mark.gpu

E_REL = 1e-10
F_ABS = 1e-8


def _dev():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device (no CPU fallback exists)"
    return torch.device("cuda", 0)


def _run(nnp, pos, types, box):
    dev = _dev()
    p = torch.tensor(np.ascontiguousarray(pos), dtype=torch.float64, device=dev)
    t = torch.tensor(np.ascontiguousarray(types), dtype=torch.int32, device=dev)
    e_atom, e_total, force = nnp.compute(p, t, box)
    torch.cuda.synchronize()
    return e_atom.cpu().numpy(), float(e_total.item()), force.cpu().numpy()


def _check_full(model, sysm, max_neighbors=None):
    """Whole-system comparison: neighbours, G, dE/dG, e_atom, E, F."""
    from paper_2002_00054_b200 import NNP
    nnp = NNP.from_model(model)
    if max_neighbors:
        nnp.set_max_neighbors(max_neighbors)
    n = sysm.n_atoms
    e_atom, e_total, force = _run(nnp, sysm.pos, sysm.types, sysm.box)
    om = oracle.OracleModel(model)
    ref = oracle.compute(om, sysm.pos, sysm.types, sysm.box)
    # neighbour sets: bit-exact
    off, idx = nnp.neighbors(n)
    roff, ridx = oracle.neighbor_list(sysm.pos, sysm.box, model.rc)
    assert np.array_equal(off.cpu().numpy(), roff)
    assert np.array_equal(idx.cpu().numpy(), ridx)
    assert np.array_equal(nnp.neighbor_counts(n).cpu().numpy(), np.diff(roff))
    # descriptors and network gradients
    G = nnp.symmetry_functions(n).cpu().numpy()
    assert np.all(np.abs(G - ref.G) <= 1e-11 * np.maximum(1.0, np.abs(ref.G)))
    B = nnp.dedg(n).cpu().numpy()
    assert np.all(np.abs(B - ref.dEdG) <= 1e-11 * np.maximum(1.0, np.abs(ref.dEdG)))
    # energies and forces
    assert np.all(np.abs(e_atom - ref.e_atom) <= 1e-10 * np.abs(ref.e_atom).max())
    assert abs(e_total - ref.e_total) <= E_REL * abs(ref.e_total)
    assert abs(e_total - e_atom.sum()) <= 1e-12 * np.abs(e_atom).sum()
    assert np.abs(force - ref.F).max() <= F_ABS
    assert np.all(np.abs(force.sum(axis=0)) < 1e-8)
    nnp.close()
    return ref


def test_config0_tiny_full_parity():
    # configs[0]: 288 atoms, L = 14.2 -> only 2 cells per dimension (periodic stencil de-dup)
    sysm, model = W.build(W.CONFIGS[0])
    ref = _check_full(model, sysm)
    assert abs(ref.e_total) > 1e-3 * np.abs(ref.e_atom).sum()     # no cancellation (reading C16)


def test_mid_size_several_cells_ragged():
    # 700 molecules -> 2100 atoms, L = 27.5 A: 4 cells per dimension, last CTAs/warps ragged
    sysm = W.make_water(700, 4242)
    _check_full(W.make_model(False), sysm)


def test_orthorhombic_box_2_3_5_cells():
    # box 12.6 x 18.7 x 31 -> 2, 3 and 5 cells: every stencil de-dup branch at once
    box = np.array([12.6, 18.7, 31.0])
    n_mol = 245
    types = np.tile(np.array([W.TYPE_O, W.TYPE_H, W.TYPE_H], dtype=np.int32), n_mol)
    sysm = W.WaterSystem(pos=_uniform_in(box, 3 * n_mol, 77), types=types, box=box, seed=77)
    _check_full(W.make_model(False), sysm)


def _uniform_in(box, n, seed):
    from workloads import rng
    k = rng.stream_key(seed, 999)
    u = rng.uniform(k, np.arange(3 * n, dtype=np.uint64)).reshape(n, 3)
    return u * box


def test_wide_model_small_system():
    sysm = W.make_water(150, 31, L=15.3)
    _check_full(W.make_model(True), sysm)


@pytest.mark.parametrize("route", ["multi", "generic"])
def test_generic_table_three_elements(route):
    # irregular table: zeta = 1, 3 and 6, Rs != 0, a missing pair group, an element with few SFs, different hidden sizes ->
    # two passes of the lane-owned kernels, exponent menus (1; 3) and (6) ("multi"), or -- with one symmetry function listed
    # twice, which no pass menu can hold -- the generic angular kernels; the generic network tiles either way
    rows = []
    for c in range(3):
        for e1 in range(3):
            rows.append((c, 2, e1, 0, 0.05 + 0.01 * c, 0.5 * e1, 0.0, 0.0))
            rows.append((c, 2, e1, 0, 0.3, 1.0, 0.0, 0.0))
        for (e1, e2) in ((0, 0), (0, 1), (1, 2), (2, 2)):      # (0,2) and (1,1) absent
            rows.append((c, 3, e1, e2, 0.002, 1.0, 3.0))
            rows.append((c, 3, e2, e1, 0.013, -1.0, 1.0))
            rows.append((c, 3, e1, e2, 0.002, -1.0, 6.0))
        if route == "generic":
            rows.append((c, 3, 0, 1, 0.002, 1.0, 3.0))
    rows = [r if len(r) == 8 else (r[0], r[1], r[2], r[3], r[4], 0.0, r[5], r[6]) for r in rows]
    model = tiny_model(rows, n_elem=3, hidden=(7, 5, 3), seed=11)
    sysm = W.make_water(120, 5, L=15.0)
    sysm.types = (np.arange(sysm.n_atoms) % 3).astype(np.int32)
    from paper_2002_00054_b200.binding import table_kernels
    assert table_kernels(model) == (route,) * 3
    _check_full(model, sysm)


@pytest.mark.parametrize("elements", [("X",), ("A", "B", "C"), ("A", "B", "C", "D")])
def test_fast_path_one_and_three_elements(elements):
    # the base-12 table on 1, 3 and 4 elements: the lane-owned kernels with a single tournament segment
    # (1 group), with 6 and with 10 pair groups (pair index derived from the slots, not from the descriptor bits);
    # 4 = NNP_MAX_ELEMENTS: every per-element array of the kernels at its full length
    model = W.make_model(False, seed=77, elements=elements, hidden=(9, 6))
    sysm = W.make_water(120, 9, L=15.0)
    sysm.types = (np.arange(sysm.n_atoms) % len(elements)).astype(np.int32)
    from paper_2002_00054_b200 import NNP
    nnp = NNP.from_model(model)
    assert nnp.uses_fast_path()
    nnp.close()
    _check_full(model, sysm)


@pytest.mark.parametrize("n_elem,n_eta", [(1, 4), (2, 4), (3, 4), (2, 2), (3, 1)])
def test_fast_path_free_eta_menu(n_elem, n_eta):
    # tables that are NOT BASELINE.json's: up to four unrelated eta values, any subset of lambda = +-1 x zeta in
    # {1, 2, 4, 16}, different subsets per pair group, one group empty -> the lane-owned kernels with per-eta
    # exponentials and missing menu entries (SpecFree32), not the generic ones
    etas = (0.0007, 0.003, 0.02, 0.0451)
    menu = ((1.0, 1.0), (-1.0, 2.0), (1.0, 4.0), (1.0, 16.0), (-1.0, 16.0), (-1.0, 1.0), (1.0, 2.0), (-1.0, 4.0))
    rows = []
    pairs = [(a, b) for a in range(n_elem) for b in range(a, n_elem)]
    for c in range(n_elem):
        for e1 in range(n_elem):
            rows.append((c, 2, e1, 0, 0.05 + 0.01 * c, 0.5 * e1, 0.0, 0.0))
            rows.append((c, 2, e1, 0, 0.3, 1.0, 0.0, 0.0))
        for ip, (e1, e2) in enumerate(pairs):
            if n_elem == 3 and ip == 2:
                continue                                     # an absent pair group
            for ie, eta in enumerate(etas[:n_eta - (c % 2 if n_eta > 2 else 0)]):   # n_eta = 4: odd elements use three only
                for im, (lam, zeta) in enumerate(menu):
                    if (im + ie + ip + c) % 3 == 0:
                        continue                             # holes in the menu, different per group and eta
                    rows.append((c, 3, e1, e2, eta, 0.0, lam, zeta))
    model = tiny_model(rows, n_elem=n_elem, hidden=(6, 4), seed=13)
    sysm = W.make_water(120, 5, L=15.0)
    sysm.types = (np.arange(sysm.n_atoms) % n_elem).astype(np.int32)
    from paper_2002_00054_b200 import NNP
    from paper_2002_00054_b200.binding import table_kernels
    assert set(table_kernels(model)) == {"free32" if n_eta > 2 else "free16"}     # <= 2 eta values: 16 accumulators
    nnp = NNP.from_model(model)
    assert nnp.uses_fast_path()
    nnp.close()
    _check_full(model, sysm)
    _check_full(model, sysm, max_neighbors=255)


def _n2p2_like_model(n_elem=2, seed=41):
    """A table shaped like published n2p2 models (not one of them): zeta in {1, 4}, lambda = +-1, seven eta values,
    angular functions of two cutoff radii, radial functions of three radii with shifts."""
    rows, rcs = [], []
    pairs = [(a, b) for a in range(n_elem) for b in range(a, n_elem)]
    for c in range(n_elem):
        for e1 in range(n_elem):
            for k, (eta, rs, rr) in enumerate(((0.003, 0.0, 6.0), (0.03, 0.0, 6.0), (0.2, 1.0, 4.5), (0.6, 2.0, 3.5))):
                rows.append((c, 2, e1, 0, eta, rs, 0.0, 0.0)); rcs.append(rr)
        for (e1, e2) in pairs:
            for ie, eta in enumerate((0.0005, 0.002, 0.004, 0.008, 0.015, 0.03, 0.07)):
                for lam in (1.0, -1.0):
                    for zeta in (1.0, 4.0):
                        if (ie + (lam > 0) + int(zeta)) % 5 == 0:
                            continue                         # holes
                        rows.append((c, 3, e1, e2, eta, 0.0, lam, zeta)); rcs.append(6.0 if ie < 5 else 4.8)
    model = tiny_model(rows, n_elem=n_elem, hidden=(12, 9), seed=seed)
    model.sf_cutoffs = rcs
    return model


@pytest.mark.parametrize("n_elem", [1, 2, 3])
def test_multi_pass_tables(n_elem):
    # more than four eta values and angular functions of several cutoff radii on the lane-owned
    # kernels, as several passes (NNP_KERNELS_MULTI) -- not on the queue-based generic ones
    from paper_2002_00054_b200 import NNP
    from paper_2002_00054_b200.binding import table_kernels
    model = _n2p2_like_model(n_elem)
    sysm = W.make_water(120, 5, L=15.0)
    sysm.types = (np.arange(sysm.n_atoms) % n_elem).astype(np.int32)
    import copy
    plain = copy.deepcopy(model); plain.sf_cutoffs = None
    assert set(table_kernels(plain)) == {"multi"}             # seven eta values: two passes even at one radius
    _check_full(plain, sysm)
    nnp = NNP.from_model(model)
    assert nnp.uses_fast_path()
    nnp.close()
    _check_full(model, sysm)                                  # + radii: 5 eta at 6.0 A (2 passes) and 2 eta at 4.8 A (1 pass)
    _check_full(model, sysm, max_neighbors=255)
    # radii on RADIAL functions only: BASELINE.json's table keeps its specialised kernels
    base = W.make_model(False)
    rc2 = np.where((base.sf["kind"] == 2) & (np.arange(len(base.sf)) % 3 == 0), 0.7 * base.rc, base.rc)
    base.sf_cutoffs = list(rc2)
    s0, _ = W.build(W.CONFIGS[0])
    _check_full(base, s0)


@pytest.mark.parametrize("zetas,kernels", [((1.0, 2.0, 4.0, 3.0), "free16"), ((2.0, 4.0, 8.0, 5.0), "free16"),
                                           ((1.0, 2.0, 3.0, 4.0, 6.0, 12.0, 48.0, 64.0), "multi")])
def test_zeta_menus(zetas, kernels):
    # any integer zeta on the lane-owned kernels: a pass carries the exponent menu {zeta0, 2 zeta0, 4 zeta0, zeta_x};
    # (1,2,4;3) and (2,4,8;5) are one pass each, the third set is the menus (1,2,4;3), (6,12;48), (64)
    from paper_2002_00054_b200.binding import table_kernels
    rows = []
    for c in range(2):
        for e1 in range(2):
            rows.append((c, 2, e1, 0, 0.05, 0.0, 0.0, 0.0))
        for (e1, e2) in ((0, 0), (0, 1), (1, 1)):
            for q, z in enumerate(zetas):
                rows.append((c, 3, e1, e2, 0.004, 0.0, 1.0, z))
                if q % 2 == 0:
                    rows.append((c, 3, e1, e2, 0.004, 0.0, -1.0, z))
                else:
                    rows.append((c, 3, e1, e2, 0.011, 0.0, -1.0, z))
    model = tiny_model(rows, n_elem=2, hidden=(6, 5), seed=41)
    assert table_kernels(model) == (kernels, kernels)
    sysm = W.make_water(150, 5, L=16.7)
    ref = _check_full(model, sysm)
    if kernels == "multi":
        # the same table in the mixed-precision mode: FP32 powers up to (1 +- cos)^64 <= 2^64 must not overflow, and no unused
        # menu entry may (0 * inf = NaN)
        from paper_2002_00054_b200 import NNP
        nnp = NNP.from_model(model)
        nnp.set_precision("mixed")
        e_atom, e_total, force = _run(nnp, sysm.pos, sysm.types, sysm.box)
        assert np.all(np.isfinite(force)) and np.all(np.isfinite(e_atom))
        assert np.abs(force - ref.F).max() < 1e-4 and abs(e_total - ref.e_total) < 1e-5 * np.abs(ref.e_atom).sum()
        nnp.close()


def test_fast_path_large_cutoff_general_exp():
    # rc = 8 A: eta_0 rc^2 = 0.064 > 0.05, so the fast kernels take the range-reduced exp (the water-like
    # configs, rc = 6 A, run on the small-argument polynomial exp_tiny)
    model = W.make_model(False, seed=5, rc=8.0)
    sysm = W.make_water(80, 13, L=16.5)
    _check_full(model, sysm)


@pytest.mark.parametrize("activation", ["softplus", "tanh"])
def test_sf_scaling_and_activation(activation):
    # model generality: affine SF scaling in front of the networks, tanh hidden layers
    import copy
    model = copy.deepcopy(W.make_model(False))
    rng = np.random.default_rng(3)
    model.sf_scaling = [(rng.uniform(0.0, 0.5, n), rng.uniform(0.2, 3.0, n)) for n in model.n_sf_per_elem]
    model.activation = activation
    sysm = W.make_water(150, 31, L=15.3)
    _check_full(model, sysm)
    # switching the scaling off again restores the plain model
    from paper_2002_00054_b200 import NNP
    nnp = NNP.from_model(model)
    for e in range(len(model.elements)):
        nnp.set_sf_scaling(e, None, None)
    nnp.set_activation("softplus")
    _, E, _ = _run(nnp, sysm.pos, sysm.types, sysm.box)
    ref = oracle.compute(oracle.OracleModel(W.make_model(False)), sysm.pos, sysm.types, sysm.box)
    assert abs(E - ref.e_total) <= E_REL * abs(ref.e_total)
    nnp.close()


def test_metal_like_small_neighbourhoods():
    # Ni-like fcc metal, rc = 3.9 A, 18 neighbours per atom -> with max_neighbors <= 64 the
    # 64-slot, one-warp-per-centre instantiation of the lane-owned kernels
    sysm, model = W.build(W.Config("fcc6", 6, False, 1, 11, 12, None, "metal"))
    _check_full(model, sysm, max_neighbors=48)
    _check_full(model, sysm)                       # and the default 160-slot kernels on the same system
    _check_full(model, sysm, max_neighbors=32)     # and the 8-lanes-per-centre kernels of k_small.cu
    _check_full(model, sysm, max_neighbors=24)     # ... with 24 slots per centre (18 neighbours fit)
    from paper_2002_00054_b200 import NNP, NNPError
    nnp = NNP.from_model(model)
    nnp.set_max_neighbors(16)                      # 18 neighbours do not fit 16: reported, not silently truncated
    with pytest.raises(NNPError) as ei:
        _run(nnp, sysm.pos, sysm.types, sysm.box)
    assert ei.value.status == 4                    # NNP_ERR_NEIGHBOR_OVERFLOW
    with pytest.raises(NNPError):
        nnp.set_max_neighbors(15)
    nnp.close()


@pytest.mark.parametrize("elements", [("X",), ("H", "O"), ("A", "B", "C")])
def test_small_neighbourhood_kernels(elements):
    # k_small.cu (max_neighbors <= 32): four centres per warp, exact pair test + compacted list; 1 - 3 elements, ragged
    # last CTA (290 atoms are not a multiple of 8), a centre without any neighbour of one element, general exp (rc = 8 would
    # not fit 32 slots, so the non-tiny variant is forced through eta instead)
    import copy
    from paper_2002_00054_b200 import NNP
    model = W.make_model(False, seed=23, rc=3.2, elements=elements, hidden=(9, 6))
    sysm = W.make_water(96, 77, L=14.2)
    sysm.types = (np.arange(sysm.n_atoms) % len(elements)).astype(np.int32)
    sysm.pos = np.concatenate([sysm.pos, [[7.1, 7.1, 7.1], [7.3, 7.0, 7.2]]])       # 290 atoms, one very close pair
    sysm.types = np.concatenate([sysm.types, [0, len(elements) - 1]]).astype(np.int32)
    nnp = NNP.from_model(model)
    nnp.set_max_neighbors(32)
    assert nnp.uses_fast_path()
    nnp.close()
    _check_full(model, sysm, max_neighbors=32)
    big = copy.deepcopy(model)                      # eta_0 rc^2 > 0.05: the range-reduced exponential
    ang = big.sf["kind"] == 3
    big.sf["eta"][ang] *= 8.0
    _check_full(big, sysm, max_neighbors=32)
    roff, _ = oracle.neighbor_list(sysm.pos, sysm.box, model.rc)
    assert 16 < np.diff(roff).max() <= 24            # at most 22 neighbours: the same cases on the 24-slot instantiation
    _check_full(model, sysm, max_neighbors=24)
    _check_full(big, sysm, max_neighbors=24)
    if len(elements) <= 2:
        # rc = 3.6 A: up to 29 neighbours; with one element 27 of the 290 centres have more than 120 contributing pairs, so their
        # lists are NOT handed from k_sf_small to k_force_small (which enumerates them itself) while their warp-mates' lists are;
        # with two elements the three groups of a centre share the 240-entry budget
        wider = W.make_model(False, seed=23, rc=3.6, elements=elements, hidden=(9, 6))
        _check_full(wider, sysm, max_neighbors=32)
    free = copy.deepcopy(model)                     # a table that is not BASELINE.json's: the lane-owned kernels, one warp per
    free.sf["eta"][ang & (free.sf["eta"] == free.sf["eta"][ang].max())] *= 1.23      # centre, rows of 24 in 64 slots
    from paper_2002_00054_b200.binding import table_kernels
    assert set(table_kernels(free)) == {"free16"}
    _check_full(free, sysm, max_neighbors=24)


def test_wide_angular_mixed_with_narrow():
    # wide angular SFs (n2p2 kind 9: no r_jk term, no r_jk cutoff) next to narrow ones in the
    # same pair group: passes of their own on the lane-owned kernels, or the generic kernels with the FP32 r_jk screen disabled
    rows = []
    for c in range(2):
        for e1 in range(2):
            rows.append((c, 2, e1, 0, 0.05, 0.0, 0.0, 0.0))
        for (e1, e2) in ((0, 0), (0, 1), (1, 1)):
            rows.append((c, 9, e1, e2, 0.004, 0.0, 1.0, 2.0))
            rows.append((c, 9, e1, e2, 0.010, 0.0, -1.0, 1.0))
            rows.append((c, 3, e1, e2, 0.004, 0.0, 1.0, 4.0))
            rows.append((c, 9, e1, e2, 0.0, 0.0, 1.0, 16.0))
    model = tiny_model(rows, n_elem=2, hidden=(5, 4), seed=21)
    from paper_2002_00054_b200.binding import table_kernels
    assert table_kernels(model) == ("multi", "multi")     # zeta in {1, 2, 4, 16}: narrow and wide passes of the lane-owned kernels
    _check_full(model, W.make_water(150, 5, L=16.7))
    _check_full(model, W.make_water(80, 21, L=12.2))      # dense: ~115 neighbours, 6,500 pairs per centre in the wide passes
    # wide only, one element, zeta = 3: a wide pass with base exponent 3; with a function listed twice: the generic kernels
    rows = [(0, 2, 0, 0, 0.05, 0.0, 0.0, 0.0), (0, 9, 0, 0, 0.02, 0.0, -1.0, 3.0), (0, 9, 0, 0, 0.001, 0.0, 1.0, 1.0)]
    sysm = W.make_water(60, 3, L=12.4)
    sysm.types[:] = 0
    assert table_kernels(tiny_model(rows, hidden=(4,), seed=3)) == ("multi",)
    _check_full(tiny_model(rows, hidden=(4,), seed=3), sysm)
    assert table_kernels(tiny_model(rows + rows[1:2], hidden=(4,), seed=3)) == ("generic",)
    _check_full(tiny_model(rows + rows[1:2], hidden=(4,), seed=3), sysm)
    # narrow and wide in one pair group on the generic kernels (a narrow function listed twice)
    _check_full(tiny_model(rows + [(0, 3, 0, 0, 0.004, 0.0, 1.0, 2.0)] * 2, hidden=(4,), seed=3), sysm)


def test_per_sf_cutoff_radii():
    # every SF with its own cutoff radius (nnp_set_sf_cutoffs) on the rc = 6 neighbourhood;
    # radial, narrow and wide angular SFs of several radii mixed in the same groups
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
    model = tiny_model(rows, n_elem=2, hidden=(5, 4), seed=31)
    model.sf_cutoffs = rcs
    _check_full(model, W.make_water(150, 5, L=16.7))
    # only ONE element of the base-52 model gets shorter radii: it moves to several passes (radial radii: generic radial-only mode), the other
    # stays on the lane-owned fast path; then back to the global rc: bit-identical to a fresh model
    from paper_2002_00054_b200 import NNP
    sysm, base = W.build(W.CONFIGS[0])
    rc2 = np.where((base.sf["central"] == 1) & (np.arange(len(base.sf)) % 3 == 0), 0.8 * base.rc, base.rc)
    base.sf_cutoffs = list(rc2)
    _check_full(base, sysm)
    nnp = NNP.from_model(base)
    nnp.set_sf_cutoffs(None)
    base.sf_cutoffs = None
    ref = NNP.from_model(base)
    a, b = _run(nnp, sysm.pos, sysm.types, sysm.box), _run(ref, sysm.pos, sysm.types, sysm.box)
    assert np.array_equal(a[0], b[0])
    nnp.close(); ref.close()


def test_sf_cutoff_argument_errors():
    from paper_2002_00054_b200 import NNP, NNPError
    model = W.make_model(False)
    nnp = NNP.from_model(model)
    n = len(model.sf)
    for bad in ([model.rc] * (n - 1), [model.rc] * (n - 1) + [model.rc * 1.01], [model.rc] * (n - 1) + [0.0],
                [model.rc] * (n - 1) + [float("nan")]):
        with pytest.raises(NNPError) as ei:
            nnp.set_sf_cutoffs(bad)
        assert ei.value.status == 1                   # NNP_ERR_INVALID_ARG
    nnp.close()


def test_n2p2_model_round_trip(tmp_path):
    # a model written as n2p2 files (fixture writer of tests/test_n2p2_reader.py), read back by
    # paper_2002_00054_b200.n2p2.read_model (SFs re-sorted, scaling / atom_energy / normalisation folded) and run on
    # the GPU: parity with the oracle on the read model, and the energy of the original model plus the offsets
    import copy
    from test_n2p2_reader import write_model
    from paper_2002_00054_b200 import NNP, n2p2
    model = copy.deepcopy(W.make_model(False))
    rs = np.random.RandomState(3)
    model.sf_scaling = [(rs.uniform(0.0, 0.5, n), rs.uniform(0.2, 3.0, n)) for n in model.n_sf_per_elem]
    model.activation = "tanh"
    offs = {"H": -0.4581, "O": -2.0413}
    write_model(str(tmp_path), model, scaling_mode="scalecenter", smin=-0.5, smax=1.5, atom_energy=offs,
                order=lambda n: list(np.random.RandomState(1).permutation(n)))
    got = n2p2.read_model(str(tmp_path))
    sysm = W.make_water(150, 31, L=15.3)
    ref_read = _check_full(got, sysm)
    ref = oracle.compute(oracle.OracleModel(model), sysm.pos, sysm.types, sysm.box)
    e_off = sum(offs[model.elements[t]] for t in sysm.types)
    assert abs(ref_read.e_total - (ref.e_total + e_off)) <= 1e-11 * abs(ref.e_total + e_off)
    nnp = NNP.from_model(got)
    assert nnp.uses_fast_path()                       # the re-sorted base-52 table still matches the base-12 shape
    nnp.close()


@pytest.mark.parametrize("wide", [False, True])
def test_mixed_precision_mode(wide):
    """the OPT-IN mixed mode (nnp_set_precision: FP32 staging and per-triplet arithmetic, FP64
    accumulation) against the same FP64 oracle, at its own measured and stated tolerance (DESIGN.md section 6c:
    max |dF| 3-6e-6 eV/A, rms 7e-7, |dE| 7e-8 of sum |E_i|) -- it does NOT meet BASELINE.json's 1e-8 / 1e-10."""
    from paper_2002_00054_b200 import NNP
    sysm = W.make_water(150, 31, L=15.3) if wide else W.make_water(700, 4242)
    model = W.make_model(wide)
    ref = oracle.compute(oracle.OracleModel(model), sysm.pos, sysm.types, sysm.box)
    nnp = NNP.from_model(model)
    nnp.set_precision("mixed")
    e_atom, e_total, force = _run(nnp, sysm.pos, sysm.types, sysm.box)
    n = sysm.n_atoms
    off, idx = nnp.neighbors(n)
    roff, ridx = oracle.neighbor_list(sysm.pos, sysm.box, model.rc)
    assert np.array_equal(off.cpu().numpy(), roff) and np.array_equal(idx.cpu().numpy(), ridx)   # the list stays FP64: bit-exact
    G = nnp.symmetry_functions(n).cpu().numpy()
    dF = np.abs(force - ref.F)
    assert 1e-9 < dF.max() <= 2e-5                     # the mode is on, and within its stated tolerance
    assert np.sqrt(np.mean(dF ** 2)) <= 3e-6
    assert np.all(np.abs(G - ref.G) <= 1e-5 * np.maximum(1.0, np.abs(ref.G)))
    assert np.abs(e_atom - ref.e_atom).max() <= 2e-5
    assert abs(e_total - ref.e_total) <= 1e-6 * np.abs(ref.e_atom).sum()
    assert np.all(np.abs(force.sum(axis=0)) < 1e-8)    # every pair term is still added to both atoms: sum F = 0
    e_atom2, e_total2, _ = _run(nnp, sysm.pos, sysm.types, sysm.box)
    assert e_total2 == e_total and np.array_equal(e_atom2, e_atom)       # energies stay bit-reproducible
    nnp.set_precision("f64")                           # and back: BASELINE.json's tolerances again
    e_atom, e_total, force = _run(nnp, sysm.pos, sysm.types, sysm.box)
    assert abs(e_total - ref.e_total) <= E_REL * abs(ref.e_total) and np.abs(force - ref.F).max() <= F_ABS
    nnp.close()


def test_single_element_radial_only():
    model = tiny_model([(0, 2, 0, 0, 0.1, 0.0, 0.0, 0.0), (0, 2, 0, 0, 0.4, 2.0, 0.0, 0.0)], hidden=(4,))
    sysm = W.make_water(60, 3, L=12.4)
    sysm.types[:] = 0
    _check_full(model, sysm)


# ------------------------------------------------------------------------ full size vs whole-system goldens
# tests/golden/fullsize_*.json are written by tests/golden/make_fullsize_golden.py from oracle/ + workloads/ alone
# (every centre of the system through the oracle, sharded over host processes): E_total, per-shard sums of E_i and F,
# an order-independent hash of every (i, j) neighbour pair per shard, projections of the whole force field, and
# row / G / E_i / F of >= 64 stratified atoms.

GOLD_DIR = os.path.join(os.path.dirname(__file__), "golden")


def _golden(cfg, call=0):
    path = os.path.join(GOLD_DIR, "fullsize_%s%s.json" % (cfg.name, "_call%d" % call if call else ""))
    assert os.path.exists(path), "missing golden %s (python tests/golden/make_fullsize_golden.py --config k)" % path
    g = json.load(open(path))
    assert g["config"] == cfg.name and g["call"] == call
    return g


def _pair_hash(i, j):
    # the digest of tests/golden/make_fullsize_golden.py: sum over pairs of a 64-bit mix of (i << 32 | j), mod 2^64
    from workloads import rng
    key = rng.stream_key(2002_00054, 0x6E6272)
    c = (i.astype(np.uint64) << np.uint64(32)) | j.astype(np.uint64)
    with np.errstate(over="ignore"):
        return int(np.add.reduce(rng.bits(key, c), dtype=np.uint64))


def _check_against_golden(g, nnp, n, e_atom, e_total, force, model, types):
    """Whole-system comparison of one evaluation with a golden file; returns a dict of the measured deviations."""
    dev = _dev()
    rep = {}
    # ---- energies: total (north_star: relative 1e-10) and per shard
    assert g["n_atoms"] == n
    rep["dE_rel"] = abs(e_total - g["e_total"]) / abs(g["e_total"])
    assert rep["dE_rel"] <= E_REL
    assert abs(g["e_total"]) > 1e-3 * g["e_abs_sum"]                    # no cancellation (reading C16)
    emax = g["e_atom_max_abs"]
    bounds = g["shards"]["bounds"]
    sh_e = np.array([math.fsum(e_atom[bounds[s]:bounds[s + 1]]) for s in range(len(bounds) - 1)])
    d = np.abs(sh_e - np.array(g["shards"]["e_sum"]))
    assert np.all(d <= 1e-10 * emax * np.maximum(np.diff(bounds), 1))
    rep["shard_dE_max"] = float(d.max())
    # ---- neighbour list of EVERY atom, bit-exact: per-shard pair counts and pair hashes
    off, idx = nnp.neighbors(n)
    off = off.cpu().numpy(); idx = idx.cpu().numpy()
    cnt = np.diff(off)
    assert int(off[-1]) == g["n_pairs"]
    assert np.array_equal(np.bincount(cnt), np.array(g["nbr_count_hist"]))
    for s in range(len(bounds) - 1):
        lo, hi = bounds[s], bounds[s + 1]
        assert int(off[hi] - off[lo]) == g["shards"]["n_pairs"][s]
        owner = np.repeat(np.arange(lo, hi, dtype=np.int64), cnt[lo:hi])
        assert "%016x" % _pair_hash(owner, idx[off[lo]:off[hi]]) == g["shards"]["nbr_hash"][s], "neighbour rows of shard %d" % s
    # ---- forces: whole-field projections, per-shard sums, net force (each bound follows from |dF| <= 1e-8 per component)
    from workloads import rng
    for k, (ref, l1) in enumerate(zip(g["force_digest"]["values"], g["force_digest"]["q_l1"])):
        q = rng.normal(rng.stream_key(g["force_digest"]["seed"], 0x646967, k), np.arange(3 * n, dtype=np.uint64)).reshape(n, 3)
        dd = abs(float(np.sum(force * q)) - ref)
        assert dd <= F_ABS * l1
        rep["digest%d_dev_over_bound" % k] = dd / (F_ABS * l1)
    sh_f = np.array([[math.fsum(force[bounds[s]:bounds[s + 1], c]) for c in range(3)] for s in range(len(bounds) - 1)])
    d = np.abs(sh_f - np.array(g["shards"]["f_sum"]))
    assert np.all(d <= F_ABS * np.maximum(np.diff(bounds), 1)[:, None])
    rep["shard_dF_max"] = float(d.max())
    assert np.all(np.abs(force.sum(axis=0)) < 1e-7)
    # ---- stratified atoms: row, G, E_i, F element by element
    atoms = np.array([a["index"] for a in g["atoms"]])
    assert len(atoms) >= 64
    G = nnp.symmetry_functions(n)[torch.tensor(atoms, device=dev)].cpu().numpy()
    dF = dG = dEa = 0.0
    for q, a in enumerate(g["atoms"]):
        m = a["index"]
        assert np.array_equal(idx[off[m]:off[m + 1]], np.array(a["row"], dtype=idx.dtype)), a["why"]
        ref_g = np.array(a["G"])
        assert ref_g.shape[0] == model.n_sf_per_elem[int(types[m])]
        gg = G[q, :ref_g.shape[0]]
        assert np.all(np.abs(gg - ref_g) <= 1e-11 * np.maximum(1.0, np.abs(ref_g))), a["why"]
        assert abs(e_atom[m] - a["e_atom"]) <= 1e-10 * emax, a["why"]
        assert np.abs(force[m] - np.array(a["F"])).max() <= F_ABS, a["why"]
        dF = max(dF, float(np.abs(force[m] - np.array(a["F"])).max()))
        dG = max(dG, float(np.abs(gg - ref_g).max()))
        dEa = max(dEa, abs(e_atom[m] - a["e_atom"]))
    rep.update(stratified_atoms=len(atoms), dF_max=dF, dG_max=dG, dEatom_max=dEa)
    return rep, off, idx


@pytest.mark.parametrize("k", [1, 2, 3, 4])
def test_full_size_configs_vs_golden(k):
    """configs[1..4] at full size, in the launch configuration bench.py times, against the whole-system oracle
    results: total energy at relative 1e-10, the neighbour list of every atom (hashes), projections and shard sums of
    the whole force field, and >= 64 stratified atoms element by element."""
    from paper_2002_00054_b200 import NNP
    cfg = W.CONFIGS[k]
    sysm, model = W.build(cfg)
    g = _golden(cfg)
    nnp = NNP.from_model(model)
    n = sysm.n_atoms
    e_atom, e_total, force = _run(nnp, sysm.pos, sysm.types, sysm.box)
    rep, off, idx = _check_against_golden(g, nnp, n, e_atom, e_total, force, model, sysm.types)
    print("full-size parity %s: %s" % (cfg.name, json.dumps(rep)))
    # properties at full size
    assert abs(e_total - e_atom.sum()) <= 1e-11 * np.abs(e_atom).sum()
    cnt = np.diff(off)
    assert 85 < cnt.mean() < 97 and cnt.max() < 160
    # neighbour symmetry j in N(i) <=> i in N(j) on a sample of rows
    for a in g["atoms"][:3]:
        m = a["index"]
        for j in idx[off[m]:off[m + 1]][:10]:
            assert m in idx[off[j]:off[j + 1]]
    # repeatability at full size (a shared-memory race in the lane-owned kernels would show up as a run-to-run
    # difference well above the reordering noise of the FP64 global atomics; compute-sanitizer is closed on this pool)
    e_atom2, e_total2, force2 = _run(nnp, sysm.pos, sysm.types, sysm.box)
    assert e_total2 == e_total and np.array_equal(e_atom2, e_atom)
    assert np.abs(force2 - force).max() < 1e-11
    nnp.close()


@pytest.mark.parametrize("max_neighbors", [24, 32])
def test_full_size_ni_like_workload_vs_golden(max_neighbors):
    """The Ni-like workload (workloads.CONFIGS[5]: 1,492,992 atoms, 18 neighbours each) at full size, in the
    launch configurations bench.py --config 5 times (the small-neighbourhood kernels of csrc/k_small.cu with 24 and with 32
    slots per centre), against the whole-system oracle results of tests/golden/fullsize_nickel1.5M.json."""
    from paper_2002_00054_b200 import NNP
    cfg = W.CONFIGS[5]
    sysm, model = W.build(cfg)
    g = _golden(cfg)
    nnp = NNP.from_model(model)
    nnp.set_max_neighbors(max_neighbors)
    n = sysm.n_atoms
    e_atom, e_total, force = _run(nnp, sysm.pos, sysm.types, sysm.box)
    rep, off, idx = _check_against_golden(g, nnp, n, e_atom, e_total, force, model, sysm.types)
    print("full-size parity %s (max_neighbors %d): %s" % (cfg.name, max_neighbors, json.dumps(rep)))
    assert abs(e_total - e_atom.sum()) <= 1e-11 * np.abs(e_atom).sum()
    cnt = np.diff(off)
    assert 17.9 < cnt.mean() < 18.1 and cnt.max() <= 24
    e_atom2, e_total2, force2 = _run(nnp, sysm.pos, sysm.types, sysm.box)
    assert e_total2 == e_total and np.array_equal(e_atom2, e_atom)
    assert np.abs(force2 - force).max() < 1e-11
    nnp.close()


def test_config1_displacement_sequence():
    """configs[1]: repeated evaluations with cumulative sigma = 0.01 A kicks (reading C15); positions
    drift out of the box and are re-wrapped by the library.  Parity at calls 0, 1, 50 (three atoms through
    oracle.forces_on) and at call 99 against the whole-system golden of that call."""
    from paper_2002_00054_b200 import NNP
    cfg = W.CONFIGS[1]
    sysm, model = W.build(cfg)
    nnp = NNP.from_model(model)
    om = oracle.OracleModel(model)
    pos = sysm.pos.copy()
    samples = np.array([5, 7777, 24575])
    for call in range(100):
        if call >= 1:
            pos = pos + W.displacement(sysm.n_atoms, cfg.seed_disp, call)
        if call in (0, 1, 50):
            e_atom, e_total, force = _run(nnp, pos, sysm.types, sysm.box)
            ref = oracle.forces_on(om, pos, sysm.types, sysm.box, samples)
            off, idx = nnp.neighbors(sysm.n_atoms)
            off = off.cpu().numpy(); idx = idx.cpu().numpy()
            for q, m in enumerate(samples):
                assert np.array_equal(idx[off[m]:off[m + 1]], ref.rows[q])
                assert abs(e_atom[m] - ref.e_atom[q]) <= 1e-10 * np.abs(e_atom).max()
                assert np.abs(force[m] - ref.F[q]).max() <= F_ABS
        elif call < 99:
            _run(nnp, pos, sysm.types, sysm.box)        # the library sees every call of the sequence
    e_atom, e_total, force = _run(nnp, pos, sysm.types, sysm.box)
    rep, _, _ = _check_against_golden(_golden(cfg, 99), nnp, sysm.n_atoms, e_atom, e_total, force, model, sysm.types)
    print("configs[1] call 99: %s" % json.dumps(rep))
    nnp.close()


# ------------------------------------------------------------------------ edge cases

def test_empty_and_tiny_inputs():
    from paper_2002_00054_b200 import NNP
    model = W.make_model(False)
    nnp = NNP.from_model(model)
    om = oracle.OracleModel(model)
    box = np.array([20.0, 20.0, 20.0])
    e_atom, e_total, force = _run(nnp, np.zeros((0, 3)), np.zeros(0, dtype=np.int32), box)
    assert e_total == 0.0 and e_atom.shape == (0,) and force.shape == (0, 3)
    # one atom: no neighbours, E = NN(0)
    pos = np.array([[3.0, 4.0, 5.0]])
    typ = np.array([1], dtype=np.int32)
    e_atom, e_total, force = _run(nnp, pos, typ, box)
    ref = oracle.compute(om, pos, typ, box)
    assert abs(e_total - ref.e_total) <= 1e-12 * abs(ref.e_total) and np.all(force == 0.0)
    # two atoms through the periodic boundary, one of them far outside the box
    pos = np.array([[0.4, 1.0, 1.0], [19.5 + 40.0, 1.0 - 20.0, 1.0]])
    typ = np.array([1, 0], dtype=np.int32)
    e_atom, e_total, force = _run(nnp, pos, typ, box)
    ref = oracle.compute(om, pos, typ, box)
    assert abs(e_total - ref.e_total) <= E_REL * abs(ref.e_total)
    assert np.abs(force - ref.F).max() <= F_ABS
    assert np.abs(force).max() > 1e-6
    nnp.close()


def test_error_codes():
    from paper_2002_00054_b200 import NNP, NNPError
    model = W.make_model(False)
    nnp = NNP.from_model(model)
    dev = _dev()
    sysm = W.make_water(50, 1, L=13.0)
    pos = torch.tensor(sysm.pos, device=dev)
    typ = torch.tensor(sysm.types, device=dev)
    with pytest.raises(NNPError) as ei:
        nnp.compute(pos, typ, [11.9, 13.0, 13.0])
    assert ei.value.status == 2                       # NNP_ERR_BOX_TOO_SMALL
    bad = typ.clone(); bad[3] = 2
    with pytest.raises(NNPError) as ei:
        nnp.compute(pos, bad, sysm.box)
    assert ei.value.status == 3                       # NNP_ERR_TYPE_RANGE
    badp = pos.clone(); badp[10, 1] = float("nan")
    with pytest.raises(NNPError) as ei:
        nnp.compute(badp, typ, sysm.box)
    assert ei.value.status == 7                       # NNP_ERR_NONFINITE
    # neighbour overflow: 150 atoms in 13^3 have ~60 neighbours each; allow only 32
    with pytest.raises(NNPError) as ei:
        nnp.set_max_neighbors(256)
    assert ei.value.status == 8                       # NNP_ERR_LIMIT (slots are addressed with 8 bits)
    nnp.set_max_neighbors(32)
    with pytest.raises(NNPError) as ei:
        nnp.compute(pos, typ, sysm.box)
    assert ei.value.status == 4                       # NNP_ERR_NEIGHBOR_OVERFLOW
    nnp.set_max_neighbors(160)
    nnp.compute(pos, typ, sysm.box)                   # recovers
    nnp.close()


def test_dense_cluster_near_max_neighbors():
    # 240 atoms in a 12.2 A box: ~115 neighbours per atom (close to the 160 cap).  Such a centre has
    # ~346 mask words, more than the workspace budget of 320 per atom: the last centres do not fit the
    # mask hand-over from k_sf2 to k_force2, so this case runs BOTH the hand-over and the force kernel's
    # own screening.
    sysm = W.make_water(80, 21, L=12.2)
    _check_full(W.make_model(False), sysm)


def test_neighbour_search_crowded_cell_sparse_grid_and_cell_limit():
    # k_neighbors runs one warp per cell on cells of rc/2 (5^3 stencil) or rc (3^3), chosen by make_grid:
    # (a) a blob that puts more than 32 atoms into one rc/2 cell: the warp walks the cell's centres in two groups of 32;
    # (b) 70 atoms in a 41 A box: fewer than 1.5 atoms per rc/2 cell -> cells of rc, and 6^3 = 216 cells exceed the
    #     workspace's cell budget of 2 n + 64 = 204, so the grid is coarsened as well (cells wider than rc);
    # (c) 1,300 atoms in a 33 x 14 x 62 A box: 10, 4 and 20 cells of rc/2 -- wrapping x-ranges, a dimension whose stencil is
    #     all of its cells, and a dimension whose interior cells skip the minimum-image test
    from workloads import rng
    model = W.make_model(False)
    sysm = W.make_water(150, 5, L=16.7)
    # 36 atoms on a jittered 4 x 3 x 3 lattice of 0.8 A inside the cell [6.68, 10.02) x [6.68, 10.02) x [3.34, 6.68) of the 5^3 grid
    # (unphysical on purpose: the arithmetic does not care, the forces get large, hence the relative force bound below)
    u = rng.uniform(rng.stream_key(31, 7), np.arange(3 * 36, dtype=np.uint64)).reshape(36, 3)
    ijk = np.array([(a, b, c) for a in range(4) for b in range(3) for c in range(3)], dtype=np.float64)
    blob = np.array([6.85, 6.85, 3.55]) + 0.8 * ijk + 0.1 * (u - 0.5)
    keep = np.ones(sysm.n_atoms, dtype=bool)
    for q in blob:                                              # drop the water atoms closer than 0.8 A to a blob atom
        d = sysm.pos - q
        d -= sysm.box * np.round(d / sysm.box)
        keep &= (d ** 2).sum(axis=1) > 0.64
    pos = np.vstack([sysm.pos[keep], blob])
    types = np.concatenate([sysm.types[keep], (np.arange(len(blob)) % 2).astype(np.int32)])
    cell = np.floor(pos / (sysm.box / 5.0)).astype(int)
    assert np.sum(np.all(cell == np.array([2, 2, 1]), axis=1)) >= 36
    from paper_2002_00054_b200 import NNP
    nnp = NNP.from_model(model)
    nnp.set_max_neighbors(200)
    e_atom, e_total, force = _run(nnp, pos, types, sysm.box)
    off, idx = nnp.neighbors(len(types))
    roff, ridx = oracle.neighbor_list(pos, sysm.box, model.rc)
    assert np.array_equal(off.cpu().numpy(), roff) and np.array_equal(idx.cpu().numpy(), ridx)
    ref = oracle.compute(oracle.OracleModel(model), pos, types, sysm.box)
    assert abs(e_total - ref.e_total) <= E_REL * np.abs(ref.e_atom).sum()
    assert np.abs(force - ref.F).max() <= F_ABS * max(1.0, np.abs(ref.F).max() / 20.0)
    nnp.close()
    for box, n, seed in ((np.array([41.0, 41.0, 41.0]), 70, 3), (np.array([33.0, 14.0, 62.0]), 1300, 4)):
        p = _uniform_in(box, n, seed)
        t = (np.arange(n) % 3 != 0).astype(np.int32)
        _check_full(model, W.WaterSystem(pos=p, types=t, box=box, seed=seed))


@pytest.mark.parametrize("max_neighbors", [128, 200])
def test_slot_capacity_variants(max_neighbors):
    # the fast kernels are instantiated for slot capacities 128 / 160 / 256 (shared-memory layout at
    # compile-time offsets); 160 is the default, these are the other two
    sysm, model = W.build(W.CONFIGS[0])
    _check_full(model, sysm, max_neighbors=max_neighbors)


def test_host_buffer_entry_point_and_determinism():
    from paper_2002_00054_b200 import NNP
    sysm, model = W.build(W.CONFIGS[0])
    nnp = NNP.from_model(model)
    e1, E1, f1 = _run(nnp, sysm.pos, sysm.types, sysm.box)
    e2, E2, f2 = _run(nnp, sysm.pos, sysm.types, sysm.box)
    assert E1 == E2 and np.array_equal(e1, e2)        # fixed summation order for energies
    assert np.abs(f1 - f2).max() < 1e-12              # forces: FP64 atomics, order may vary
    eh, Eh, fh = nnp.compute_host(sysm.pos, sysm.types, sysm.box)
    assert Eh[0] == E1 and np.array_equal(eh, e1) and np.abs(fh - f1).max() < 1e-12
    nnp.close()


def test_timings_and_launch_count():
    from paper_2002_00054_b200 import NNP
    sysm, model = W.build(W.CONFIGS[0])
    nnp = NNP.from_model(model)
    nnp.set_timing(True)
    _run(nnp, sysm.pos, sysm.types, sysm.box)
    t = nnp.timings_ms()
    assert set(t) == {"sort", "neighbors", "symmetry_functions", "networks", "forces", "finalize"}
    assert all(v >= 0.0 for v in t.values()) and t["forces"] > 0.0
    assert nnp.last_launch_count() >= 9
    nnp.close()


@pytest.mark.parametrize("which", ["water-fast", "metal-small", "generic"])
def test_deterministic_forces(which):
    # nnp_set_deterministic_forces: fixed-point (2^-40 eV/A) global accumulation -> the SAME BITS on every run (the default
    # FP64 atomics repeat to ~1e-13 only), still within BASELINE.json's 1e-8 of the oracle
    from paper_2002_00054_b200 import NNP
    kw = {}
    if which == "water-fast":
        sysm, model = W.build(W.CONFIGS[1])                      # 24,576 atoms: thousands of CTAs racing on the atomics
    elif which == "metal-small":
        sysm, model = W.build(W.Config("fcc10", 10, False, 1, 11, 12, None, "metal"))
        kw["max_neighbors"] = 32
    else:
        rows = []
        for c in range(2):
            for e1 in range(2):
                rows.append((c, 2, e1, 0, 0.05, 0.0, 0.0, 0.0))
            for (e1, e2) in ((0, 0), (0, 1), (1, 1)):
                rows.append((c, 3, e1, e2, 0.004, 0.0, 1.0, 3.0))
                rows.append((c, 9, e1, e2, 0.010, 0.0, -1.0, 1.0))
            rows.append(rows[-1])                                # listed twice: no pass menu holds it -> the generic kernels
        model = tiny_model(rows, n_elem=2, hidden=(5, 4), seed=21)
        from paper_2002_00054_b200.binding import table_kernels
        assert table_kernels(model) == ("generic", "generic")
        sysm = W.make_water(700, 4242)
    nnp = NNP.from_model(model)
    if "max_neighbors" in kw:
        nnp.set_max_neighbors(kw["max_neighbors"])
    nnp.set_deterministic_forces(True)
    runs = [_run(nnp, sysm.pos, sysm.types, sysm.box) for _ in range(3)]
    for r in runs[1:]:
        assert np.array_equal(r[2], runs[0][2]) and np.array_equal(r[0], runs[0][0]) and r[1] == runs[0][1]
    assert np.all(np.abs(runs[0][2].sum(axis=0)) < 1e-7)
    nnp.set_deterministic_forces(False)
    plain = _run(nnp, sysm.pos, sysm.types, sysm.box)
    assert np.abs(plain[2] - runs[0][2]).max() < 1e-10            # ~180 contributions per atom, each rounded to 9.1e-13
    if sysm.n_atoms <= 5000:
        ref = oracle.compute(oracle.OracleModel(model), sysm.pos, sysm.types, sysm.box)
    else:
        g = _golden(W.CONFIGS[1])
        ref = None
        for a in g["atoms"]:
            assert np.abs(runs[0][2][a["index"]] - np.array(a["F"])).max() <= F_ABS
    if ref is not None:
        assert np.abs(runs[0][2] - ref.F).max() <= F_ABS
    nnp.close()


def test_deterministic_forces_range_error():
    # a neighbour 1e-9 A from the centre: the 1/a factors of the angular force terms exceed the fixed-point range
    from paper_2002_00054_b200 import NNP, NNPError
    model = W.make_model(False)
    nnp = NNP.from_model(model)
    nnp.set_deterministic_forces(True)
    pos = np.array([[5.0, 5.0, 5.0], [5.0 + 1e-9, 5.0, 5.0], [7.0, 6.0, 5.0], [4.0, 7.0, 6.5]])
    typ = np.array([1, 0, 0, 1], dtype=np.int32)
    dev = _dev()
    with pytest.raises(NNPError) as ei:
        nnp.compute(torch.tensor(pos, device=dev), torch.tensor(typ, device=dev), [20.0, 20.0, 20.0])
    assert ei.value.status == 9                       # NNP_ERR_FORCE_RANGE
    nnp.close()
