"""CPU oracle of the MD loop around the path (TEST INFRASTRUCTURE ONLY, like the rest of oracle/).

Velocity Verlet, NVE, written out step by step (the paper checks its
implementation by energy conservation):
    v(t + dt/2) = v(t) + (dt/2) a(t)          a = ACC_UNIT * F / m
    x(t + dt)   = x(t) + dt v(t + dt/2)
    F(t + dt)   = forces of the NNP at x(t + dt)            (oracle.compute: O(N^2) neighbours)
    v(t + dt)   = v(t + dt/2) + (dt/2) a(t + dt)
Units: A, eV, amu, fs.  ACC_UNIT converts eV/(A amu) to A/fs^2:
    1 eV/A = 1.602176634e-19 J / 1e-10 m, 1 amu = 1.66053906660e-27 kg, 1 m/s^2 = 1e10 A / 1e30 fs^2
    -> ACC_UNIT = (1.602176634e-19 / 1e-10) / 1.66053906660e-27 * 1e10 / 1e30 = 9.648533215665327e-3.
Pins (tests/test_oracle_md_pins.py): the constant from CODATA values, time reversibility, energy error
falling 4x when dt is halved, momentum conservation.  Positions are not wrapped (the force routine wraps).
"""
from __future__ import annotations

import numpy as np

from . import compute

ACC_UNIT = (1.602176634e-19 / 1e-10) / 1.66053906660e-27 * 1e10 / 1e30


def kinetic_energy(vel, types, masses):
    m = np.asarray(masses, dtype=np.float64)[np.asarray(types)]
    return float(np.sum(m * np.sum(np.asarray(vel, dtype=np.float64) ** 2, axis=1)) / (2.0 * ACC_UNIT))


def run(om, pos, vel, types, box, masses, dt, n_steps):
    """Returns (pos, vel, F, e_pot list incl. step 0, e_kin list incl. step 0)."""
    x = np.array(pos, dtype=np.float64)
    v = np.array(vel, dtype=np.float64)
    m = np.asarray(masses, dtype=np.float64)[np.asarray(types)][:, None]
    r = compute(om, x, types, box)
    F = r.F
    epot, ekin = [r.e_total], [kinetic_energy(v, types, masses)]
    for _ in range(n_steps):
        v = v + (0.5 * dt) * ACC_UNIT * F / m
        x = x + dt * v
        r = compute(om, x, types, box)
        F = r.F
        v = v + (0.5 * dt) * ACC_UNIT * F / m
        epot.append(r.e_total)
        ekin.append(kinetic_energy(v, types, masses))
    return x, v, F, epot, ekin
