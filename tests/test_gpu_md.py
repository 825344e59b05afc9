"""MD loop around the path: the CUDA velocity-Verlet loop (nnp_md_run, nnp_md_kinetic_energy)
against the CPU oracle (oracle/md.py) step for step, and the check the paper itself uses for its
implementation -- energy conservation of an NVE run."""
import numpy as np
import pytest
import torch

import oracle
import workloads as W
from oracle import md

pytestmark = pytest.mark.gpu
MASS = (1.008, 15.999)


def _state(sysm, seed, sigma=0.005):
    rng = np.random.default_rng(seed)
    vel = rng.normal(0.0, sigma, size=(sysm.n_atoms, 3))
    m = np.asarray(MASS)[sysm.types][:, None]
    vel -= (m * vel).sum(axis=0) / m.sum()
    return vel


def test_md_trajectory_matches_oracle():
    from paper_2002_00054_b200 import NNP
    sysm, model = W.build(W.CONFIGS[0])
    vel = _state(sysm, 3)
    dev = torch.device("cuda", 0)
    nnp = NNP.from_model(model)
    pos_d = torch.tensor(sysm.pos, dtype=torch.float64, device=dev)
    vel_d = torch.tensor(vel, dtype=torch.float64, device=dev)
    typ_d = torch.tensor(sysm.types, dtype=torch.int32, device=dev)
    state = nnp.compute(pos_d, typ_d, sysm.box)
    ek0 = float(nnp.kinetic_energy(MASS, vel_d, typ_d).item())
    assert abs(ek0 - md.kinetic_energy(vel, sysm.types, MASS)) < 1e-12 * ek0
    n_steps, dt = 8, 0.5
    nnp.md_run(n_steps, dt, MASS, pos_d, vel_d, typ_d, sysm.box, state)
    x, v, F, ep, ek = md.run(oracle.OracleModel(model), sysm.pos, vel, sysm.types, sysm.box, MASS, dt, n_steps)
    assert np.abs(pos_d.cpu().numpy() - x).max() < 1e-9
    assert np.abs(vel_d.cpu().numpy() - v).max() < 1e-10
    assert np.abs(state[2].cpu().numpy() - F).max() < 1e-8
    assert abs(float(state[1].item()) - ep[-1]) < 1e-10 * abs(ep[-1])
    assert abs(float(nnp.kinetic_energy(MASS, vel_d, typ_d).item()) - ek[-1]) < 1e-9 * ek[-1]
    nnp.close()


def test_md_energy_conservation_nve():
    # 2,100 atoms, 300 steps of 0.25 fs: the total energy must not drift (forces consistent with the energy)
    from paper_2002_00054_b200 import NNP
    sysm = W.make_water(700, 4242)
    model = W.make_model(False)
    vel = _state(sysm, 9)
    dev = torch.device("cuda", 0)
    nnp = NNP.from_model(model)
    pos_d = torch.tensor(sysm.pos, dtype=torch.float64, device=dev)
    vel_d = torch.tensor(vel, dtype=torch.float64, device=dev)
    typ_d = torch.tensor(sysm.types, dtype=torch.int32, device=dev)
    state = nnp.compute(pos_d, typ_d, sysm.box)
    e = []
    for _ in range(6):
        e.append(float(state[1].item()) + float(nnp.kinetic_energy(MASS, vel_d, typ_d).item()))
        nnp.md_run(50, 0.25, MASS, pos_d, vel_d, typ_d, sysm.box, state)
    e.append(float(state[1].item()) + float(nnp.kinetic_energy(MASS, vel_d, typ_d).item()))
    e = np.array(e)
    ekin = float(nnp.kinetic_energy(MASS, vel_d, typ_d).item())
    assert np.abs(e - e[0]).max() < 2e-3 * ekin          # fluctuation of the Verlet shadow energy, no drift
    assert abs(e[-1] - e[0]) < 2e-3 * ekin
    nnp.close()


def test_md_argument_errors():
    from paper_2002_00054_b200 import NNP, NNPError
    sysm, model = W.build(W.CONFIGS[0])
    dev = torch.device("cuda", 0)
    nnp = NNP.from_model(model)
    pos_d = torch.tensor(sysm.pos, dtype=torch.float64, device=dev)
    vel_d = torch.zeros_like(pos_d)
    typ_d = torch.tensor(sysm.types, dtype=torch.int32, device=dev)
    state = nnp.compute(pos_d, typ_d, sysm.box)
    with pytest.raises(NNPError):
        nnp.md_run(1, -1.0, MASS, pos_d, vel_d, typ_d, sysm.box, state)
    with pytest.raises(NNPError):
        nnp.md_run(1, 0.5, (1.0, 0.0), pos_d, vel_d, typ_d, sysm.box, state)
    nnp.md_run(0, 0.5, MASS, pos_d, vel_d, typ_d, sysm.box, state)     # zero steps: nothing changes
    assert torch.equal(pos_d.cpu(), torch.tensor(sysm.pos, dtype=torch.float64))
    nnp.close()


def _imploding_shell():
    """One centre atom and 33 atoms on a sphere of radius 8.5 A around it, flying inwards at 1 A/fs: with
    max_neighbors = 32 the start (radius 8.5) and the end (radius 7.5 on the far side, 16 fs later) are fine, the
    steps in between overflow (33 neighbours of the centre at radius < 6, all 33 mutual below ~3).  The shell
    passes the centre between two steps (radius 0.5 -> -0.5), so no two atoms ever coincide."""
    k = np.arange(33) + 0.5
    phi = np.arccos(1.0 - 2.0 * k / 33.0)
    th = np.pi * (1.0 + 5.0 ** 0.5) * k
    unit = np.stack([np.cos(th) * np.sin(phi), np.sin(th) * np.sin(phi), np.cos(phi)], axis=1)
    c = np.array([20.0, 20.0, 20.0])
    pos = np.concatenate([[c], c + 8.5 * unit])
    vel = np.concatenate([[np.zeros(3)], -1.0 * unit])
    types = np.zeros(34, dtype=np.int32)
    return pos, vel, types, np.array([40.0, 40.0, 40.0])


@pytest.mark.parametrize("n_steps", [16, 3])     # 16: CUDA-graph replay of steps 2..n; 3: plain launches
def test_md_run_reports_an_error_of_a_middle_step(n_steps):
    # every step's nnp_compute clears the device status word, so an overflow in steps 5..11 used to be
    # lost (NNP_OK after the run, wrong forces integrated).  The sticky word keeps it until nnp_sync_status.
    from paper_2002_00054_b200 import NNP, NNPError
    model = W.make_model(False, seed=5, elements=("X",), hidden=(6, 4))
    pos, vel, types, box = _imploding_shell()
    dev = torch.device("cuda", 0)
    nnp = NNP.from_model(model)
    nnp.set_max_neighbors(32)
    pos_d = torch.tensor(pos, dtype=torch.float64, device=dev)
    vel_d = torch.tensor(vel, dtype=torch.float64, device=dev)
    typ_d = torch.tensor(types, dtype=torch.int32, device=dev)
    heavy = (1.0e6,)                                   # ballistic: the forces do not deflect anything
    state = nnp.compute(pos_d, typ_d, box)             # radius 8.5: fine
    with pytest.raises(NNPError) as ei:                # 16 steps of 1 fs, or 3 steps of 16/3 fs (radius 8.5, 3.17, -2.17, -7.5)
        nnp.md_run(n_steps, 16.0 / n_steps, heavy, pos_d, vel_d, typ_d, box, state)
    assert ei.value.status == 4                        # NNP_ERR_NEIGHBOR_OVERFLOW, from a middle step
    r = np.linalg.norm(pos_d.cpu().numpy()[1:] - pos[0], axis=1)
    assert np.all(np.abs(r - 7.5) < 1e-3)              # the LAST step is fine again
    nnp.compute(pos_d, typ_d, box)                     # ... and reading cleared the sticky word
    nnp.close()


def test_sync_status_covers_every_call_since_the_last_sync():
    from paper_2002_00054_b200 import NNP, NNPError
    sysm, model = W.build(W.CONFIGS[0])
    dev = torch.device("cuda", 0)
    nnp = NNP.from_model(model)
    good = torch.tensor(sysm.pos, dtype=torch.float64, device=dev)
    bad = good.clone(); bad[17, 2] = float("inf")
    typ = torch.tensor(sysm.types, dtype=torch.int32, device=dev)
    nnp.compute(good, typ, sysm.box, sync=False)
    nnp.compute(bad, typ, sysm.box, sync=False)
    nnp.compute(good, typ, sysm.box, sync=False)
    with pytest.raises(NNPError) as ei:
        nnp.sync_status()
    assert ei.value.status == 7                        # NNP_ERR_NONFINITE of the middle call
    nnp.sync_status()                                  # cleared by reading
    nnp.close()
