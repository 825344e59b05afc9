"""Invariances of the CUDA path itself ("translational, rotational, and permutational ... are included in the
descriptors"), checked on the GPU output directly -- not through the oracle, which has its own
copies of these tests.  Energies to the rounding of a re-ordered FP64 sum, forces transformed accordingly."""
import numpy as np
import pytest
import torch

import workloads as W

pytestmark = pytest.mark.gpu


def _eval(nnp, pos, types, box):
    dev = torch.device("cuda", 0)
    p = torch.tensor(np.ascontiguousarray(pos), dtype=torch.float64, device=dev)
    t = torch.tensor(np.ascontiguousarray(types), dtype=torch.int32, device=dev)
    e_atom, e_total, force = nnp.compute(p, t, box)
    torch.cuda.synchronize()
    return e_atom.cpu().numpy(), float(e_total.item()), force.cpu().numpy()


@pytest.fixture(scope="module")
def setup():
    from paper_2002_00054_b200 import NNP
    sysm = W.make_water(700, 4242)                      # 2,100 atoms, 4 cells per dimension
    model = W.make_model(False)
    nnp = NNP.from_model(model)
    ref = _eval(nnp, sysm.pos, sysm.types, sysm.box)
    yield nnp, sysm, ref
    nnp.close()


def test_translation_and_lattice_shift(setup):
    nnp, sysm, (e_atom, E, F) = setup
    for shift in (np.array([0.37, -1.91, 5.55]), sysm.box * np.array([1.0, -2.0, 3.0]), np.array([1e3, 1e3, -1e3])):
        ea, E2, F2 = _eval(nnp, sysm.pos + shift, sysm.types, sysm.box)
        tol = 1e-11 if np.abs(shift).max() < 100 else 1e-8          # a 1,000 A shift costs 1e-13 A of coordinate precision
        assert abs(E2 - E) <= tol * abs(E)
        assert np.abs(ea - e_atom).max() <= tol * np.abs(e_atom).max()
        assert np.abs(F2 - F).max() <= 1e3 * tol * max(1.0, np.abs(F).max())


def test_cube_rotations_and_mirror(setup):
    nnp, sysm, (e_atom, E, F) = setup
    # the 48 cube symmetries = signed axis permutations; a cubic periodic box maps onto itself
    for perm, signs in (((1, 2, 0), (1, 1, 1)), ((2, 0, 1), (-1, 1, -1)), ((1, 0, 2), (1, -1, 1)), ((0, 1, 2), (-1, -1, -1))):
        Rm = np.zeros((3, 3))
        for r in range(3):
            Rm[r, perm[r]] = signs[r]
        ea, E2, F2 = _eval(nnp, sysm.pos @ Rm.T, sysm.types, sysm.box[list(perm)])
        assert abs(E2 - E) <= 1e-11 * abs(E)
        assert np.abs(ea - e_atom).max() <= 1e-11 * np.abs(e_atom).max()
        assert np.abs(F2 - F @ Rm.T).max() <= 1e-9


def test_same_element_permutation(setup):
    nnp, sysm, (e_atom, E, F) = setup
    rs = np.random.RandomState(7)
    perm = np.arange(sysm.n_atoms)
    for t in (0, 1):                                     # shuffle the atoms of every element among themselves
        idx = np.flatnonzero(sysm.types == t)
        perm[idx] = rs.permutation(idx)
    ea, E2, F2 = _eval(nnp, sysm.pos[perm], sysm.types[perm], sysm.box)
    assert abs(E2 - E) <= 1e-11 * abs(E)
    assert np.abs(ea - e_atom[perm]).max() <= 1e-11 * np.abs(e_atom).max()
    assert np.abs(F2 - F[perm]).max() <= 1e-9
    # any permutation (types move with the atoms)
    perm = rs.permutation(sysm.n_atoms)
    ea, E2, F2 = _eval(nnp, sysm.pos[perm], sysm.types[perm], sysm.box)
    assert abs(E2 - E) <= 1e-11 * abs(E) and np.abs(F2 - F[perm]).max() <= 1e-9


def test_forces_are_the_gradient_of_the_energy(setup):
    # central finite differences of the GPU energy against the GPU forces, h = 1e-4 A (relative 1e-6: O(h^2) truncation)
    nnp, sysm, (e_atom, E, F) = setup
    rs = np.random.RandomState(11)
    h = 1e-4
    for m in rs.choice(sysm.n_atoms, 4, replace=False):
        for c in range(3):
            p = sysm.pos.copy(); p[m, c] += h
            Ep = _eval(nnp, p, sysm.types, sysm.box)[1]
            p[m, c] -= 2 * h
            Em = _eval(nnp, p, sysm.types, sysm.box)[1]
            fd = -(Ep - Em) / (2 * h)
            assert abs(fd - F[m, c]) <= 1e-6 * max(1.0, abs(F[m, c])) + 5e-7     # + cancellation noise of E ~ 1e4 eV / h
