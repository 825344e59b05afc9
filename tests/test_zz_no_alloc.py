"""nnp_md_kinetic_energy_noalloc -- the entry point that allocates nothing (its block sums sit in a static device array
inside the library, csrc/k_noalloc.cu) -- against the existing nnp_md_kinetic_energy, which keeps them in the caller's
workspace.  Same arithmetic and summation order, so the comparison could be exact; the bound used is the one
tests/test_gpu_md.py uses for the kinetic energy (1e-12 relative).  Two calls in a row, the second on a smaller system
and other velocities: the array keeps the first call's block sums, and the second result must not see them.

This file is named to be collected LAST (the suite runs with pytest -x)."""
import numpy as np
import pytest
import torch

import workloads as W

pytestmark = pytest.mark.gpu
MASS = (1.008, 15.999)
REL = 1e-12


def _inputs(sysm, seed, sigma, dev):
    rng = np.random.default_rng(seed)
    vel = rng.normal(0.0, sigma, size=(sysm.n_atoms, 3))
    return (torch.tensor(vel, dtype=torch.float64, device=dev),
            torch.tensor(sysm.types, dtype=torch.int32, device=dev), vel)


def test_kinetic_energy_noalloc_matches_workspace_path_twice():
    from paper_2002_00054_b200 import NNP
    dev = torch.device("cuda", 0)
    model = W.make_model(False)
    nnp = NNP.from_model(model)
    big = W.make_water(700, 4242)            # 2,100 atoms: 9 block sums, the last block ragged
    small = W.make_water(150, 5, L=16.7)     # 450 atoms: 2 block sums -- 7 stale ones stay behind in the array
    out = torch.full((1,), float("nan"), dtype=torch.float64, device=dev)      # caller-owned result buffer
    for sysm, seed, sigma in ((big, 3, 0.01), (small, 4, 0.02)):
        vel_d, typ_d, vel = _inputs(sysm, seed, sigma, dev)
        ref = float(nnp.kinetic_energy(MASS, vel_d, typ_d).item())              # existing path (workspace scratch)
        before = torch.cuda.memory_allocated(dev)
        nnp.kinetic_energy_noalloc(MASS, vel_d, typ_d, out)
        torch.cuda.synchronize()
        assert torch.cuda.memory_allocated(dev) == before
        got = float(out.item())
        assert ref > 0.0
        assert abs(got - ref) <= REL * ref
        # and both against the plain definition sum m v^2 / (2 NNP_ACC_UNIT)
        acc_unit = 9.648533215665327e-3
        m = np.asarray(MASS)[sysm.types]
        plain = float((m * (vel ** 2).sum(axis=1)).sum() / (2.0 * acc_unit))
        assert abs(got - plain) <= 1e-11 * plain
    # empty system: E_kin = 0, nothing read
    vel_d, typ_d, _ = _inputs(small, 5, 0.01, dev)
    nnp.kinetic_energy_noalloc(MASS, vel_d, typ_d, out, n_atoms=0)
    torch.cuda.synchronize()
    assert float(out.item()) == 0.0
    nnp.close()


def test_kinetic_energy_noalloc_rejects_sizes_beyond_the_static_array():
    from paper_2002_00054_b200 import NNP, NNPError
    dev = torch.device("cuda", 0)
    nnp = NNP.from_model(W.make_model(False))
    sysm = W.make_water(150, 5, L=16.7)
    vel_d, typ_d, _ = _inputs(sysm, 6, 0.01, dev)
    out = torch.full((1,), -1.0, dtype=torch.float64, device=dev)
    with pytest.raises(NNPError) as ei:      # checked before anything is launched: the small buffers are never read
        nnp.kinetic_energy_noalloc(MASS, vel_d, typ_d, out, n_atoms=4194304 + 1)
    assert "LIMIT" in str(ei.value).upper() and "NNP_NOALLOC_MAX_ATOMS" in str(ei.value)
    torch.cuda.synchronize()
    assert float(out.item()) == -1.0
    with pytest.raises(NNPError):
        nnp.kinetic_energy_noalloc((1.0, -2.0), vel_d, typ_d, out)
    nnp.close()
