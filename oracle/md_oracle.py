"""Velocity-Verlet MD loop of the CPU oracle.

TEST INFRASTRUCTURE -- same rule as oracle.py: only tests/, smoke() and bench.py's cpu_baseline / reference legs may
import this.  Plain numpy, fp64, one statement per step of the scheme, forces from oracle.evaluate.

PAPER.md:151-153 (section VI-A): "the MD equations are numerically integrated by the velocity-Verlet scheme for 500
steps (the energy and forces are evaluated for 501 times) at time-steps of 0.5 fs (water) and 1.0 fs (copper)".
The paper names the scheme and gives no formula; velocity Verlet is the textbook one:
    v(t + dt/2) = v(t) + (dt/2) a(t);   x(t + dt) = x(t) + dt v(t + dt/2);   a(t + dt) = F(x(t + dt)) / m;
    v(t + dt) = v(t + dt/2) + (dt/2) a(t + dt).
Units: Angstrom, fs, amu, eV.  1 (eV/A)/amu = e / amu * 1e-10 A/fs^2 (CODATA 2018 exact e, 2018 amu).
Pins (tests/test_oracle_md.py): free flight with a zero-weight model, time reversibility, momentum conservation,
total-energy error falling as dt^2, the unit constant against scipy.constants.
"""
from __future__ import annotations

import numpy as np

from . import oracle

E_CHARGE = 1.602176634e-19          # C
AMU = 1.66053906660e-27             # kg
ACC = E_CHARGE / AMU * 1.0e-10      # A/fs^2 per (eV/A)/amu


def kinetic_energy(vel: np.ndarray, mass_per_atom: np.ndarray) -> float:
    """sum_i 1/2 m_i |v_i|^2 in eV (v in A/fs, m in amu)."""
    return float(np.sum(0.5 * mass_per_atom[:, None] * vel * vel) / ACC)


def run(coords, vel, types, masses, box, model, dt_fs: float, nsteps: int, force_fn=None):
    """Returns dict(coords, vel, forces, thermo [nsteps+1, 2] = (E_pot, E_kin), virial of the last evaluation)."""
    ev = force_fn if force_fn is not None else (lambda x: oracle.evaluate(x, types, box, model))
    x = np.array(coords, dtype=np.float64, copy=True)
    v = np.array(vel, dtype=np.float64, copy=True)
    m = np.asarray(masses, dtype=np.float64)[np.asarray(types)]
    thermo = np.zeros((nsteps + 1, 2))
    o = ev(x)
    f = o["forces"]
    thermo[0] = (o["energy"], kinetic_energy(v, m))
    for s in range(1, nsteps + 1):
        a = f / m[:, None] * ACC
        v = v + 0.5 * dt_fs * a
        x = x + dt_fs * v
        o = ev(x)
        f = o["forces"]
        a = f / m[:, None] * ACC
        v = v + 0.5 * dt_fs * a
        thermo[s] = (o["energy"], kinetic_energy(v, m))
    return dict(coords=x, vel=v, forces=f, thermo=thermo, virial=o["virial"])
