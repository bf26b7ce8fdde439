"""Velocity-Verlet MD loop of the CPU oracle.

TEST INFRASTRUCTURE -- same rule as oracle.py: only tests/, smoke() and bench.py's cpu_baseline / reference legs may
import this.  Plain numpy, fp64, one statement per step of the scheme, forces from oracle.evaluate.

PAPER.md:151-153 (section VI-A): "the MD equations are numerically integrated by the velocity-Verlet scheme for 500
steps (the energy and forces are evaluated for 501 times) at time-steps of 0.5 fs (water) and 1.0 fs (copper)".
The paper names the scheme and gives no formula; velocity Verlet is the textbook one:
    v(t + dt/2) = v(t) + (dt/2) a(t);   x(t + dt) = x(t) + dt v(t + dt/2);   a(t + dt) = F(x(t + dt)) / m;
    v(t + dt) = v(t + dt/2) + (dt/2) a(t + dt).
Units: Angstrom, fs, amu, eV.  1 (eV/A)/amu = e / amu * 1e-10 A/fs^2 (CODATA 2018 exact e, 2018 amu).
Thermodynamic record ("kinetic energy, potential energy, temperature, pressure, are collected"; the paper
gives no formula, these are the textbook ones, LAMMPS' conventions): T = 2 KE / ((3 N - 3) kB) (three conserved momentum
components removed from the degrees of freedom), P = (2 KE + trace(Xi)) / (3 V) with Xi = -dE/d(strain) the virial of
DESIGN.md reading Q18, in bar (1 eV/A^3 = 1.602176634e6 bar).
Pins (tests/test_oracle_md.py): free flight with a zero-weight model, time reversibility, momentum conservation,
total-energy error falling as dt^2, the unit constants against scipy.constants, the ideal-gas law P V = (N - 1) kB T for a
zero-weight model, T near the 330 K of the seeded Boltzmann velocities, P = -dE/dV by a finite volume change at rest.
"""
from __future__ import annotations

import numpy as np

from . import oracle

E_CHARGE = 1.602176634e-19          # C
AMU = 1.66053906660e-27             # kg
ACC = E_CHARGE / AMU * 1.0e-10      # A/fs^2 per (eV/A)/amu
KB = 8.617333262e-5                 # eV/K (CODATA 2018)
EV_A3_TO_BAR = E_CHARGE * 1.0e30 * 1.0e-5   # 1 eV/A^3 in bar


def kinetic_energy(vel: np.ndarray, mass_per_atom: np.ndarray) -> float:
    """sum_i 1/2 m_i |v_i|^2 in eV (v in A/fs, m in amu)."""
    return float(np.sum(0.5 * mass_per_atom[:, None] * vel * vel) / ACC)


def temperature(ke: float, natoms: int) -> float:
    """T = 2 KE / ((3 N - 3) kB) in K."""
    dof = 3.0 * natoms - 3.0 if natoms > 1 else 3.0
    return 2.0 * ke / (dof * KB)


def pressure(ke: float, virial: np.ndarray, box: np.ndarray) -> float:
    """P = (2 KE + trace(Xi)) / (3 V) in bar; V = |det(box)|."""
    vol = abs(float(np.linalg.det(np.asarray(box, dtype=np.float64).reshape(3, 3))))
    v = np.asarray(virial, dtype=np.float64).reshape(9)
    return (2.0 * ke + v[0] + v[4] + v[8]) / (3.0 * vol) * EV_A3_TO_BAR


def run(coords, vel, types, masses, box, model, dt_fs: float, nsteps: int, force_fn=None):
    """Returns dict(coords, vel, forces, thermo [nsteps+1, 4] = (E_pot, E_kin, T, P), virial of the last evaluation)."""
    ev = force_fn if force_fn is not None else (lambda x: oracle.evaluate(x, types, box, model))
    x = np.array(coords, dtype=np.float64, copy=True)
    v = np.array(vel, dtype=np.float64, copy=True)
    m = np.asarray(masses, dtype=np.float64)[np.asarray(types)]
    thermo = np.zeros((nsteps + 1, 4))
    n = x.shape[0]

    def record(o, v):
        ke = kinetic_energy(v, m)
        return (o["energy"], ke, temperature(ke, n), pressure(ke, o["virial"], box))

    o = ev(x)
    f = o["forces"]
    thermo[0] = record(o, v)
    for s in range(1, nsteps + 1):
        a = f / m[:, None] * ACC
        v = v + 0.5 * dt_fs * a
        x = x + dt_fs * v
        o = ev(x)
        f = o["forces"]
        a = f / m[:, None] * ACC
        v = v + 0.5 * dt_fs * a
        thermo[s] = record(o, v)
    return dict(coords=x, vel=v, forces=f, thermo=thermo, virial=o["virial"])
