"""dp_md_run (velocity-Verlet loop) against the MD oracle, through the C ABI (-m gpu)."""
import numpy as np
import pytest

from oracle import md_oracle
from paper_2005_00223_b200 import synth

pytestmark = pytest.mark.gpu


def _gpu_md(s, v, masses, dt, nsteps, precision, skin=0.0, rebuild_every=0, want_status=False):
    import torch
    from paper_2005_00223_b200 import binding
    m = binding.DPModel(s.model, precision)
    c = torch.from_numpy(s.coords.copy()).cuda()
    vel = torch.from_numpy(v.copy()).cuda()
    t = torch.from_numpy(s.types).cuda()
    out = m.md_run(c, vel, t, masses, s.box, dt, nsteps, skin=skin, rebuild_every=rebuild_every)
    rc, _ = m.status()
    if want_status:
        m.close()
        return rc
    assert rc == 0
    torch.cuda.synchronize()
    res = {k: x.cpu().numpy() for k, x in out.items()}
    res["nlist"] = m.get_nlist().cpu().numpy()
    res["coords"], res["vel"] = c.cpu().numpy(), vel.cpu().numpy()
    m.close()
    return res


@pytest.mark.parametrize("idx,dt,nsteps", [(0, 1.0, 6), (1, 0.5, 4)])      # copper 1.0 fs, water 0.5 fs
def test_md_trajectory_fp64_matches_oracle(idx, dt, nsteps):
    s = synth.config(idx)
    masses = synth.MASS_AMU["cu" if idx == 0 else "water"]
    v = synth.boltzmann_velocities(s.types, masses, 330.0, 4242 + idx)
    o = md_oracle.run(s.coords, v, s.types, masses, s.box, s.model, dt, nsteps)
    g = _gpu_md(s, v, masses, dt, nsteps, "fp64")
    assert np.abs(g["coords"] - o["coords"]).max() <= 1e-11
    vr = np.sqrt((o["vel"] ** 2).mean())
    assert np.abs(g["vel"] - o["vel"]).max() <= 1e-10 * vr
    fr = np.sqrt((o["forces"] ** 2).mean())
    assert np.abs(g["forces"] - o["forces"]).max() <= 1e-9 * fr       # forces at positions that differ by rounding
    assert np.abs(g["thermo"][:, 0] - o["thermo"][:, 0]).max() <= 1e-12 * abs(o["thermo"][0, 0])
    assert np.abs(g["thermo"][:, 1] - o["thermo"][:, 1]).max() <= 1e-11 * o["thermo"][0, 1]
    # temperature and pressure of every evaluation; the pressure carries the virial of that evaluation
    assert np.abs(g["thermo"][:, 2] - o["thermo"][:, 2]).max() <= 1e-10 * o["thermo"][0, 2]
    assert np.abs(g["thermo"][:, 3] - o["thermo"][:, 3]).max() <= 1e-9 * np.abs(o["thermo"][:, 3]).max()
    assert np.abs(g["virial"] - o["virial"]).max() <= 1e-9 * np.abs(o["virial"]).max()
    assert np.abs(o["coords"] - s.coords).max() > 1e-3


def test_md_zero_steps_is_one_evaluation_and_bad_arguments():
    import torch
    from paper_2005_00223_b200 import binding
    s = synth.config(0)
    v = synth.boltzmann_velocities(s.types, (63.546,), 330.0, 1)
    g = _gpu_md(s, v, (63.546,), 1.0, 0, "fp64")
    assert np.array_equal(g["coords"], s.coords) and np.array_equal(g["vel"], v)
    assert g["thermo"].shape == (1, 4)
    m = binding.DPModel(s.model, "fp64")
    c = torch.from_numpy(s.coords.copy()).cuda(); vel = torch.from_numpy(v.copy()).cuda(); t = torch.from_numpy(s.types).cuda()
    for masses, dt, n in [((0.0,), 1.0, 1), ((63.5,), 0.0, 1), ((63.5,), 1.0, -1)]:
        with pytest.raises(binding.DPError) as e:
            m.md_run(c, vel, t, masses, s.box, dt, n)
        assert e.value.code == -1
    m.close()


def test_md_mix16_conserves_total_energy():
    # the benchmark precision on config 0's geometry: 20 steps of 1 fs; the total energy must stay put far better than
    # its parts move (mixed-precision forces are not exactly conservative: bound the drift, PAPER.md:127 discusses it)
    s = synth.config(0)
    masses = (1.0,)                                                   # light atoms so that the dynamics matter in 20 fs
    v = synth.boltzmann_velocities(s.types, masses, 30.0, 7)
    g = _gpu_md(s, v, masses, 1.0, 20, "mix16")
    e = g["thermo"][:, 0] + g["thermo"][:, 1]
    moved = np.ptp(g["thermo"][:, 1])
    assert moved > 0 and np.abs(e - e[0]).max() < 0.05 * moved, (np.abs(e - e[0]).max(), moved)


@pytest.mark.parametrize("idx,dt,nsteps,every", [(0, 1.0, 7, 3), (1, 0.5, 5, 4), (0, 1.0, 6, 3)])
def test_md_buffered_list_gives_the_same_trajectory_and_list(idx, dt, nsteps, every):
    # 2 A buffer; list searches at evaluations 0, every, 2 every, ...; the steps between re-test the stored
    # candidates.  The formatted list of the LAST evaluation (a reuse step in the first two cases, a search in the third)
    # must still be the oracle's, bit for bit.
    from oracle import oracle
    s = synth.config(idx)
    masses = synth.MASS_AMU["cu" if idx == 0 else "water"]
    v = synth.boltzmann_velocities(s.types, masses, 330.0, 4242 + idx)
    o = md_oracle.run(s.coords, v, s.types, masses, s.box, s.model, dt, nsteps)
    g = _gpu_md(s, v, masses, dt, nsteps, "fp64", skin=2.0, rebuild_every=every)
    assert np.abs(g["coords"] - o["coords"]).max() <= 1e-11
    assert np.abs(g["vel"] - o["vel"]).max() <= 1e-10 * np.sqrt((o["vel"] ** 2).mean())
    assert np.abs(g["thermo"][:, 0] - o["thermo"][:, 0]).max() <= 1e-12 * abs(o["thermo"][0, 0])
    fin = oracle.evaluate(g["coords"], s.types, s.box, s.model)
    assert np.array_equal(g["nlist"], fin["nlist"])
    fr = np.sqrt((fin["forces"] ** 2).mean())
    assert np.abs(g["forces"] - fin["forces"]).max() <= 1e-10 * fr


def test_md_buffered_list_reports_an_atom_that_outran_the_buffer():
    s = synth.config(0)
    v = synth.boltzmann_velocities(s.types, (63.546,), 330.0, 1)
    v[17] = [0.3, 0.0, 0.0]                      # 0.3 A/fs: 1.5 A after 5 fs, beyond half of a 2 A buffer
    assert _gpu_md(s, v, (63.546,), 1.0, 5, "fp64", skin=2.0, rebuild_every=50, want_status=True) == -8
    assert _gpu_md(s, v, (63.546,), 1.0, 2, "fp64", skin=2.0, rebuild_every=50, want_status=True) == 0
    # the flags of ALL evaluations of a run are reported: the atom outruns the buffer at evaluation 4, the run ends on a
    # search (evaluation 6 = 2 x 3), whose own flags are clean
    v[17] = [0.4, 0.0, 0.0]
    assert _gpu_md(s, v, (63.546,), 1.0, 6, "fp64", skin=2.0, rebuild_every=6, want_status=True) == -8


def test_md_buffered_list_reports_candidate_overflow_of_an_earlier_search():
    # skin 3 A: 298 candidates within rc + skin = 9.5 A... against the 512-entry candidate store this fits; use sel = 16 so
    # that the store holds 256: the search of evaluation 0 overflows (DP_ENEIGH) and the later reuse steps must not hide it
    s = synth.copper(6, 0.05, 3, sel=(16,))
    v = synth.boltzmann_velocities(s.types, (63.546,), 330.0, 1)
    assert _gpu_md(s, v, (63.546,), 1.0, 3, "fp64", skin=1.6, rebuild_every=50, want_status=True) == -6


def test_md_buffered_list_mix16_matches_unbuffered_energies():
    s = synth.config(0)
    masses = (1.0,)
    v = synth.boltzmann_velocities(s.types, masses, 30.0, 7)
    a = _gpu_md(s, v, masses, 1.0, 12, "mix16")
    b = _gpu_md(s, v, masses, 1.0, 12, "mix16", skin=2.0, rebuild_every=5)
    swing = np.ptp(a["thermo"][:, 1])
    assert np.abs(a["thermo"][:, :2] - b["thermo"][:, :2]).max() < 1e-3 * swing
    # the list of the buffered run's last evaluation (a reuse step) is the oracle's list at that run's own final coordinates
    from oracle import oracle
    fin = oracle.evaluate(b["coords"], s.types, s.box, s.model)
    assert np.array_equal(b["nlist"], fin["nlist"])
