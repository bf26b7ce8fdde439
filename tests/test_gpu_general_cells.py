"""SURVEY.md 8(f)-3 through the C ABI (-m gpu): boxes shorter than 2 rc, triclinic cells (explicit ghost images, ghost.cu),
more than two atom types.  Same bars as test_gpu_parity.py: list bit-exact, FP64 1e-12 / 1e-10, MIX-32 1e-4, MIX-16 5e-3."""
import numpy as np
import pytest

from oracle import oracle
from paper_2005_00223_b200 import synth

pytestmark = pytest.mark.gpu


def _gpu_eval(coords, types, box, model, precision):
    import torch
    from paper_2005_00223_b200 import binding
    m = binding.DPModel(model, precision)
    out = m.compute(torch.from_numpy(np.ascontiguousarray(coords)).cuda(), torch.from_numpy(types).cuda(), box)
    rc, ntr = m.status()
    assert rc == 0, rc
    nl = m.get_nlist()
    torch.cuda.synchronize()
    res = {k: v.cpu().numpy() for k, v in out.items()}
    res["nlist"] = nl.cpu().numpy()
    res["n_truncated"] = ntr
    m.close()
    return res


def _check(g, o, prec, natoms):
    tolF = {"fp64": 1e-10, "mix32": 1e-4, "mix16": 5e-3}[prec]
    assert np.array_equal(g["nlist"], o["nlist"])
    assert g["n_truncated"] == o["n_truncated"]
    rms = np.sqrt((o["forces"] ** 2).mean())
    err = np.abs(g["forces"] - o["forces"]).max()
    assert err <= tolF * rms, (prec, err / rms)
    vmax = np.abs(o["virial"]).max()
    assert np.abs(g["virial"] - o["virial"]).max() <= tolF * vmax, (prec, np.abs(g["virial"] - o["virial"]).max() / vmax)
    if prec == "fp64":
        assert abs(g["energy"][0] - o["energy"]) <= 1e-12 * abs(o["energy"])
        assert np.abs(g["atom_energy"] - o["atom_energy"]).max() <= 1e-11 * np.abs(o["atom_energy"]).max()
    else:
        assert abs(g["energy"][0] - o["energy"]) / natoms <= (2e-5 if prec == "mix32" else 1e-3)
    assert np.abs(g["forces"].sum(0)).max() <= 1e-6 * max(np.abs(g["forces"]).sum(0).max(), 1e-30)


def _rot(seed):
    rng = np.random.default_rng(seed)
    q, r = np.linalg.qr(rng.standard_normal((3, 3)))
    q = q * np.sign(np.diag(r))
    if np.linalg.det(q) < 0:
        q[:, 0] = -q[:, 0]
    return q


@pytest.mark.parametrize("prec", ["fp64", "mix32", "mix16"])
def test_box_shorter_than_two_rc_multiple_images(prec):
    """32 atoms, two types, L = 7.27 A < 2 rc = 8.4 A: an atom sees two images of some neighbours"""
    s = synth.small_fcc(2, 41, sigma=0.08, rc=4.2, rc_smth=1.2, sel=(48,), ntypes=2)
    o = oracle.evaluate(s.coords, s.types, s.box, s.model)
    _check(_gpu_eval(s.coords, s.types, s.box, s.model, prec), o, prec, s.natoms)


def test_very_small_box_two_images_per_axis_and_exact_ties():
    """4 atoms of an ideal lattice in a box of ONE FCC cell, L = 3.634 A, rc = 5 A: image range 2 per axis; equal distances
    everywhere (several images of one atom share a key): the list (user indices) and E, F, virial are still the oracle's"""
    s = synth.small_fcc(1, 3, sigma=0.0, rc=5.0, rc_smth=1.5, sel=(96,))
    o = oracle.evaluate(s.coords, s.types, s.box, s.model)
    assert o["n_truncated"] == 0 and (o["nlist"] >= 0).sum(axis=1).min() == 42       # three FCC shells, all images
    g = _gpu_eval(s.coords, s.types, s.box, s.model, "fp64")
    assert np.array_equal(g["nlist"], o["nlist"])
    assert abs(g["energy"][0] - o["energy"]) <= 1e-12 * abs(o["energy"])
    assert np.abs(g["forces"] - o["forces"]).max() <= 1e-12                # a perfect lattice: zero force
    assert np.abs(g["virial"] - o["virial"]).max() <= 1e-10 * np.abs(o["virial"]).max()


def test_sheared_cell_random_atoms(prec="fp64"):
    rng = np.random.default_rng(3)
    H = np.array([[6.2, 0.0, 0.0], [1.9, 5.8, 0.0], [0.7, -1.4, 6.5]])
    n = 60
    x = rng.random((n, 3)) @ H + rng.integers(-2, 3, size=(n, 3)) @ H          # also atoms outside the cell
    types = (np.arange(n) % 2).astype(np.int32)
    m = synth.make_model(2, 4.0, 1.0, (64, 64), 77, [[0.1, 0, 0, 0]] * 2, [[0.2, 0.15, 0.15, 0.15]] * 2)
    o = oracle.evaluate(x, types, H.reshape(9), m)
    _check(_gpu_eval(x, types, H.reshape(9), m, prec), o, prec, n)


@pytest.mark.parametrize("prec", ["fp64", "mix32", "mix16"])
def test_rechosen_sheared_cell_of_a_two_type_lattice(prec):
    """108 atoms, two types, the cell a' = a + b, c' = c + a - b of a cubic lattice: a sheared cell with short heights"""
    s = synth.small_fcc(3, 9, sigma=0.06, rc=4.5, rc_smth=1.0, sel=(40, 40), ntypes=2)
    box = (np.array([[1, 1, 0], [0, 1, 0], [1, -1, 1]]) @ s.box.reshape(3, 3)).reshape(9).astype(np.float64)
    o = oracle.evaluate(s.coords, s.types, box, s.model)
    _check(_gpu_eval(s.coords, s.types, box, s.model, prec), o, prec, s.natoms)


@pytest.mark.parametrize("prec", ["fp64", "mix16"])
def test_rotated_config0_is_a_triclinic_cell_with_long_edges(prec):
    """config 0 (copper 500 atoms, L = 18.17 >= 2 rc) rotated: a general cell -> ghost path with one image per axis"""
    s = synth.config(0)
    Q = _rot(7)
    x = s.coords @ Q
    box = (s.box.reshape(3, 3) @ Q).reshape(9)
    o = oracle.evaluate(x, s.types, box, s.model)
    _check(_gpu_eval(x, s.types, box, s.model, prec), o, prec, s.natoms)


@pytest.mark.parametrize("ntypes", [3, 4])
@pytest.mark.parametrize("prec", ["fp64", "mix32", "mix16"])
def test_three_and_four_atom_types(ntypes, prec):
    """the multi-component systems of PAPER.md:107: T^2 embedding nets, T fitting nets, T neighbour blocks per row"""
    s = synth.small_fcc(4, 50 + ntypes, sigma=0.08, rc=5.0, rc_smth=1.5, sel=(24,), ntypes=ntypes)     # 256 atoms, L = 14.5
    o = oracle.evaluate(s.coords, s.types, s.box, s.model)
    _check(_gpu_eval(s.coords, s.types, s.box, s.model, prec), o, prec, s.natoms)


def test_three_types_in_a_small_sheared_cell():
    rng = np.random.default_rng(9)
    H = np.array([[5.5, 0.0, 0.0], [-1.2, 5.9, 0.0], [1.4, 0.9, 5.1]])
    n = 40
    x = rng.random((n, 3)) @ H
    types = (np.arange(n) % 3).astype(np.int32)
    m = synth.make_model(3, 4.5, 1.0, (48, 48, 48), 5, [[0.1, 0, 0, 0]] * 3, [[0.2, 0.15, 0.15, 0.15]] * 3)
    o = oracle.evaluate(x, types, H.reshape(9), m)
    _check(_gpu_eval(x, types, H.reshape(9), m, "fp64"), o, "fp64", n)


def test_sixteen_types_are_accepted_and_seventeen_are_not():
    from paper_2005_00223_b200 import binding
    s = synth.small_fcc(3, 8, sigma=0.05, rc=4.0, rc_smth=1.0, sel=(4,), ntypes=16)      # 108 atoms, L = 10.9
    o = oracle.evaluate(s.coords, s.types, s.box, s.model)
    _check(_gpu_eval(s.coords, s.types, s.box, s.model, "fp64"), o, "fp64", s.natoms)
    m17 = synth.make_model(17, 4.0, 1.0, (4,) * 17, 1, [[0.1, 0, 0, 0]] * 17, [[0.2, 0.1, 0.1, 0.1]] * 17)
    with pytest.raises(binding.DPError) as e:
        binding.DPModel(m17, "fp64")
    assert e.value.code == -1


def test_md_in_a_small_box_matches_the_md_oracle():
    from oracle import md_oracle
    import torch
    from paper_2005_00223_b200 import binding
    s = synth.small_fcc(2, 77, sigma=0.08, rc=3.6, rc_smth=1.0, sel=(24,), ntypes=2)       # 32 atoms, multi-image box
    masses = (63.546, 26.98)
    v = synth.boltzmann_velocities(s.types, masses, 330.0, 5)
    o = md_oracle.run(s.coords, v, s.types, masses, s.box, s.model, 1.0, 3)
    m = binding.DPModel(s.model, "fp64")
    c, vel, t = torch.from_numpy(s.coords.copy()).cuda(), torch.from_numpy(v.copy()).cuda(), torch.from_numpy(s.types).cuda()
    g = m.md_run(c, vel, t, masses, s.box, 1.0, 3, skin=2.0, rebuild_every=50)     # the buffer is ignored in ghost mode
    rc, _ = m.status()
    assert rc == 0
    assert np.abs(c.cpu().numpy() - o["coords"]).max() <= 1e-11
    th = g["thermo"].cpu().numpy()
    assert np.abs(th[:, 0] - o["thermo"][:, 0]).max() <= 1e-12 * abs(o["thermo"][0, 0])
    assert np.abs(th[:, 3] - o["thermo"][:, 3]).max() <= 1e-9 * np.abs(o["thermo"][:, 3]).max()
    m.close()
