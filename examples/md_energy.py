"""Energy-conservation table of an NVE run (the check the paper uses for its own
implementation, PAPER.md L80 / Suppl. S2): `python examples/md_energy.py [--molecules M] [--fs T]`.

For each time step dt the same start state is integrated for T fs with `nnp_md_run` (velocity Verlet on the
device, neighbour list rebuilt every step) and the total energy E = E_pot + E_kin is sampled; forces that are
the exact gradient of the energy give a bounded fluctuation of E that shrinks as dt^2 and no drift.
Prints a markdown table; every number comes from the CUDA path (no oracle, no CPU fallback).
"""
import argparse
import os
import sys

import numpy as np
import torch

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))

import workloads as W
from paper_2002_00054_b200 import NNP

MASS = (1.008, 15.999)          # amu, element order ("H", "O") of workloads.make_model


def run(n_mol, t_fs, dts, samples, seed, sigma):
    sysm = W.make_water(n_mol, seed)
    model = W.make_model(False)
    rng = np.random.default_rng(seed + 1)
    vel = rng.normal(0.0, sigma, size=(sysm.n_atoms, 3))
    m = np.asarray(MASS)[sysm.types][:, None]
    vel -= (m * vel).sum(axis=0) / m.sum()
    dev = torch.device("cuda", 0)
    nnp = NNP.from_model(model)
    typ_d = torch.tensor(sysm.types, dtype=torch.int32, device=dev)
    rows = []
    for dt in dts:
        pos_d = torch.tensor(sysm.pos, dtype=torch.float64, device=dev)
        vel_d = torch.tensor(vel, dtype=torch.float64, device=dev)
        state = nnp.compute(pos_d, typ_d, sysm.box)
        n_steps = int(round(t_fs / dt))
        chunk = max(1, n_steps // samples)
        e, ek = [], []
        done = 0
        while True:
            k = float(nnp.kinetic_energy(MASS, vel_d, typ_d).item())
            ek.append(k)
            e.append(float(state[1].item()) + k)
            if done >= n_steps:
                break
            s = min(chunk, n_steps - done)
            nnp.md_run(s, dt, MASS, pos_d, vel_d, typ_d, sysm.box, state)
            done += s
        e, ek = np.array(e), np.array(ek)
        t = np.linspace(0.0, done * dt, len(e))
        slope = np.polyfit(t, e, 1)[0]
        rows.append((dt, done, e[0], np.abs(e - e[0]).max(), e.std(), slope * 1000.0 / sysm.n_atoms, ek.mean()))
    nnp.close()
    return sysm.n_atoms, rows


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--molecules", type=int, default=8192)
    ap.add_argument("--fs", type=float, default=100.0)
    ap.add_argument("--dt", type=float, nargs="+", default=[0.5, 0.25, 0.125])
    ap.add_argument("--samples", type=int, default=50)
    ap.add_argument("--seed", type=int, default=4242)
    ap.add_argument("--sigma", type=float, default=0.005, help="initial velocity spread, A/fs")
    a = ap.parse_args()
    n, rows = run(a.molecules, a.fs, a.dt, a.samples, a.seed, a.sigma)
    print(f"NVE, {n} atoms, {a.fs} fs per run, water-like synthetic system and base-52 model (workloads/), "
          f"{torch.cuda.get_device_name(0)}")
    print()
    print("| dt (fs) | steps | E(0) (eV) | max abs(E - E(0)) (eV) | std E (eV) | std E / mean E_kin | drift (meV/atom/ps) | mean E_kin (eV) |")
    print("|---|---|---|---|---|---|---|---|")
    for dt, steps, e0, dmax, sd, drift, ek in rows:
        print(f"| {dt:g} | {steps} | {e0:.6f} | {dmax:.3e} | {sd:.3e} | {sd / ek:.2e} | {drift:+.3e} | {ek:.4f} |")
    if len(rows) >= 2:
        print()
        for (d1, _, _, _, s1, _, _), (d2, _, _, _, s2, _, _) in zip(rows[:-1], rows[1:]):
            print(f"std E ratio dt={d1:g} / dt={d2:g}: {s1 / s2:.2f} (dt^2 scaling: {(d1 / d2) ** 2:.2f})")


if __name__ == "__main__":
    main()
