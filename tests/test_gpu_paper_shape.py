"""SURVEY.md 8(f)-2 through the C ABI (-m gpu): the paper's own network shape, embedding nets (32, 64, 128), neighbour
capacities 512 (copper) / 144 (water), on the config-0 / config-1 geometries, against the oracle."""
import numpy as np
import pytest

from oracle import oracle
from paper_2005_00223_b200 import synth

pytestmark = pytest.mark.gpu


def _gpu_eval(s, precision):
    import torch
    from paper_2005_00223_b200 import binding
    m = binding.DPModel(s.model, precision)
    out = m.compute(torch.from_numpy(s.coords).cuda(), torch.from_numpy(s.types).cuda(), s.box)
    rc, ntr = m.status()
    assert rc == 0, rc
    nl = m.get_nlist()
    torch.cuda.synchronize()
    res = {k: v.cpu().numpy() for k, v in out.items()}
    res["nlist"] = nl.cpu().numpy()
    res["n_truncated"] = ntr
    m.close()
    return res


def _systems():
    return [synth.paper_copper(5, 20200510), synth.paper_water(512, 24.83, 20200511)]


@pytest.mark.parametrize("k", [0, 1])
def test_paper_shape_fp64(k):
    s = _systems()[k]
    o = oracle.evaluate(s.coords, s.types, s.box, s.model)
    g = _gpu_eval(s, "fp64")
    assert np.array_equal(g["nlist"], o["nlist"]) and g["n_truncated"] == o["n_truncated"]
    assert abs(g["energy"][0] - o["energy"]) <= 1e-12 * abs(o["energy"])
    assert np.abs(g["atom_energy"] - o["atom_energy"]).max() <= 1e-11 * np.abs(o["atom_energy"]).max()
    rms = np.sqrt((o["forces"] ** 2).mean())
    assert np.abs(g["forces"] - o["forces"]).max() <= 1e-10 * rms
    assert np.abs(g["virial"] - o["virial"]).max() <= 1e-10 * np.abs(o["virial"]).max()


@pytest.mark.parametrize("k", [0, 1])
def test_paper_shape_mix16(k):
    """MIX-16 at the paper's shape (tcgen05 kernels templated on the width; biases through the constant-ones K step)"""
    s = _systems()[k]
    o = oracle.evaluate(s.coords, s.types, s.box, s.model)
    g = _gpu_eval(s, "mix16")
    assert np.array_equal(g["nlist"], o["nlist"]) and g["n_truncated"] == o["n_truncated"]
    rms = np.sqrt((o["forces"] ** 2).mean())
    err = np.abs(g["forces"] - o["forces"]).max()
    assert err <= 5e-3 * rms, err / rms
    assert abs(g["energy"][0] - o["energy"]) / s.natoms <= 1e-3
    assert np.abs(g["atom_energy"] - o["atom_energy"]).max() <= 5e-3
    assert np.abs(g["virial"] - o["virial"]).max() / s.natoms <= 1e-3


def test_paper_shape_mix32_water():
    """MIX-32 at the paper's shape on the water geometry (the north_star MIX-32 bound, 1e-4 RMS(F), is stated for water)"""
    s = _systems()[1]
    o = oracle.evaluate(s.coords, s.types, s.box, s.model)
    g = _gpu_eval(s, "mix32")
    assert np.array_equal(g["nlist"], o["nlist"]) and g["n_truncated"] == o["n_truncated"]
    rms = np.sqrt((o["forces"] ** 2).mean())
    err = np.abs(g["forces"] - o["forces"]).max()
    assert err <= 1e-4 * rms, err / rms
    assert abs(g["energy"][0] - o["energy"]) / s.natoms <= 2e-5
    assert np.abs(g["virial"] - o["virial"]).max() / s.natoms <= 2e-5


def test_paper_shape_mix32_copper():
    """MIX-32 at the paper's shape on the copper geometry: bounded as in test_copper_mix32_and_mix16_parity_config2_geometry
    (the paper's own MIX-32 RMS force deviation, and the MIX-16 relative bound)"""
    s = _systems()[0]
    o = oracle.evaluate(s.coords, s.types, s.box, s.model)
    g = _gpu_eval(s, "mix32")
    assert np.array_equal(g["nlist"], o["nlist"])
    dF = g["forces"] - o["forces"]
    rms = np.sqrt((o["forces"] ** 2).mean())
    assert np.sqrt((dF ** 2).mean()) <= 2.5e-6 and np.abs(dF).max() <= 5e-3 * rms, (np.sqrt((dF ** 2).mean()), np.abs(dF).max() / rms)
    assert abs(g["energy"][0] - o["energy"]) / s.natoms <= 2e-5
