"""Pins of the MD oracle (oracle/md_oracle.py, velocity Verlet) against what the mathematics fixes:
free flight, time reversibility, momentum conservation, total-energy error ~ dt^2, the unit constant.  CPU only."""
import numpy as np
import scipy.constants as sc

from oracle import md_oracle
from paper_2005_00223_b200 import synth


def _fcc():
    s = synth.small_fcc(2, 77, sigma=0.08, rc=3.6, rc_smth=1.0, sel=(24,), ntypes=2)      # 32 atoms, multi-image box
    masses = (63.546, 26.98)
    v = synth.boltzmann_velocities(s.types, masses, 330.0, 5)
    return s, masses, v


def test_unit_constant_against_codata():
    # 1 (eV/A)/amu = e / (amu * 1e-10 m) m/s^2 = ... * 1e10 A / (1e15 fs)^2
    acc = sc.e / (sc.atomic_mass * 1e-10) * 1e10 / 1e30
    assert abs(md_oracle.ACC - acc) <= 1e-8 * acc            # CODATA 2018 vs the scipy release's amu
    assert abs(md_oracle.ACC - 9.648533216e-3) < 1e-11
    # kinetic energy of one 12-amu atom at 1 A/fs = 0.5 * 12 amu * (1e5 m/s)^2 in eV
    ke = 0.5 * 12 * sc.atomic_mass * (1e5) ** 2 / sc.e
    assert abs(md_oracle.kinetic_energy(np.array([[1.0, 0.0, 0.0]]), np.array([12.0])) - ke) <= 1e-8 * ke


def test_boltzmann_generator_temperature_and_momentum():
    types = np.zeros(20000, dtype=np.int32)
    v = synth.boltzmann_velocities(types, (63.546,), 330.0, 1)
    m = np.full(20000, 63.546)
    T = 2.0 * md_oracle.kinetic_energy(v, m) / (3 * 20000 * sc.k / sc.e)
    assert abs(T - 330.0) < 5.0
    assert np.abs((m[:, None] * v).sum(0)).max() < 1e-9


def test_free_flight_with_zero_weights():
    s, masses, v = _fcc()
    z = synth.make_model(2, s.model.rc, s.model.rc_smth, s.model.sel, 1, s.model.avg, s.model.std, zero=True)
    r = md_oracle.run(s.coords, v, s.types, masses, s.box, z, 0.7, 5)
    assert np.abs(r["coords"] - (s.coords + 3.5 * v)).max() < 1e-13
    assert np.array_equal(r["vel"], v)
    assert np.all(r["thermo"][:, 0] == r["thermo"][0, 0]) and np.ptp(r["thermo"][:, 1]) == 0.0


def test_time_reversibility_and_momentum():
    s, masses, v = _fcc()
    a = md_oracle.run(s.coords, v, s.types, masses, s.box, s.model, 1.0, 6)
    b = md_oracle.run(a["coords"], -a["vel"], s.types, masses, s.box, s.model, 1.0, 6)
    assert np.abs(b["coords"] - s.coords).max() < 1e-11
    assert np.abs(b["vel"] + v).max() < 1e-12
    m = np.asarray(masses)[s.types]
    assert np.abs((m[:, None] * a["vel"]).sum(0)).max() < 1e-10       # started at zero total momentum
    assert np.abs(a["coords"] - s.coords).max() > 1e-3                 # something moved


def test_one_step_matches_hand_expansion():
    # x(dt) = x + dt v + dt^2/2 a(x) exactly for velocity Verlet; a from the oracle's forces at x
    from oracle import oracle
    s, masses, v = _fcc()
    dt = 0.5
    f0 = oracle.evaluate(s.coords, s.types, s.box, s.model)["forces"]
    m = np.asarray(masses)[s.types][:, None]
    r = md_oracle.run(s.coords, v, s.types, masses, s.box, s.model, dt, 1)
    x1 = s.coords + dt * v + 0.5 * dt * dt * f0 / m * (sc.e / sc.atomic_mass * 1e-10)
    assert np.abs(r["coords"] - x1).max() < 1e-12
    f1 = oracle.evaluate(x1, s.types, s.box, s.model)["forces"]
    v1 = v + 0.5 * dt * (f0 + f1) / m * (sc.e / sc.atomic_mass * 1e-10)
    assert np.abs(r["vel"] - v1).max() < 1e-12


def test_total_energy_error_scales_as_dt_squared():
    # light atoms so that 16 fs of dynamics moves several eV between potential and kinetic energy
    s, _, _ = _fcc()
    masses = (1.0, 0.6)
    v = synth.boltzmann_velocities(s.types, masses, 30.0, 9)

    def dev(dt, n):
        th = md_oracle.run(s.coords, v, s.types, masses, s.box, s.model, dt, n)["thermo"]
        e = th[:, 0] + th[:, 1]
        return np.abs(e - e[0]).max(), np.ptp(th[:, 1])
    d1, k1 = dev(2.0, 8)
    d2, _ = dev(1.0, 16)
    assert k1 > 50 * d1            # the total is conserved far better than its parts move
    assert 2.5 < d1 / d2 < 6.0, (d1, d2)


def test_temperature_and_pressure_record():
    """PAPER.md:153 thermo record.  Unit constants against scipy; ideal-gas law for a zero-weight model (Xi = 0):
    P V = (N - 1) kB T; T of the seeded 330 K velocities; the potential part of P equals -dE/dV by a finite isotropic
    volume change at rest (uses the oracle's virial, pinned separately by strain finite differences)."""
    from oracle import oracle
    assert abs(md_oracle.KB - sc.k / sc.e) < 1e-13            # 8.617333262e-5 eV/K is the 10-digit CODATA value
    assert abs(md_oracle.EV_A3_TO_BAR - sc.e * 1e30 / 1e5) < 1e-6
    s, masses, v = _fcc()
    z = synth.make_model(2, s.model.rc, s.model.rc_smth, s.model.sel, 1, s.model.avg, s.model.std, zero=True)
    th = md_oracle.run(s.coords, v, s.types, masses, s.box, z, 0.5, 2)["thermo"]
    n = s.natoms
    vol = s.box[0] * s.box[4] * s.box[8]
    assert np.allclose(th[:, 3] * 1e5 * vol * 1e-30, (n - 1) * sc.k * th[:, 2], rtol=1e-9)     # Pa m^3 = J
    big = synth.boltzmann_velocities(np.zeros(30000, dtype=np.int32), (63.546,), 330.0, 3)
    ke = md_oracle.kinetic_energy(big, np.full(30000, 63.546))
    assert abs(md_oracle.temperature(ke, 30000) - 330.0) < 4.0
    # potential pressure at rest: -dE/dV with V -> V (1 + 3 h): coordinates and box scaled by (1 + h)
    h = 1e-5
    ep = oracle.evaluate(s.coords * (1 + h), s.types, s.box * (1 + h), s.model)["energy"]
    em = oracle.evaluate(s.coords * (1 - h), s.types, s.box * (1 - h), s.model)["energy"]
    p_fd = -(ep - em) / (vol * ((1 + h) ** 3 - (1 - h) ** 3)) * md_oracle.EV_A3_TO_BAR
    o = oracle.evaluate(s.coords, s.types, s.box, s.model)
    p_or = md_oracle.pressure(0.0, o["virial"], s.box)
    assert abs(p_or - p_fd) <= 1e-6 * max(abs(p_fd), 1.0), (p_or, p_fd)
