"""GPU vs oracle parity through the C ABI (-m gpu).

Tolerances (BASELINE.json north_star): neighbour list bit-exact; FP64 |dE|/|E| <= 1e-12 and
max|dF| <= 1e-10 * RMS(F_oracle); virial: same relative tolerance against max|Xi|.
"""
import numpy as np
import pytest

from oracle import oracle
from paper_2005_00223_b200 import synth

pytestmark = pytest.mark.gpu


def _gpu_eval(s, precision=None):
    import torch
    from paper_2005_00223_b200 import binding
    m = binding.DPModel(s.model, precision or s.precision)
    c = torch.from_numpy(s.coords).cuda()
    t = torch.from_numpy(s.types).cuda()
    out = m.compute(c, t, s.box)
    rc, ntr = m.status()
    assert rc == 0, rc
    nl = m.get_nlist()
    torch.cuda.synchronize()
    res = {k: v.cpu().numpy() for k, v in out.items()}
    res["nlist"] = nl.cpu().numpy()
    res["n_truncated"] = ntr
    res["rows"] = m.last_row_counts()
    m.close()
    return res


def _check_fp64(g, o, tolE=1e-12, tolF=1e-10):
    assert np.array_equal(g["nlist"], o["nlist"])
    assert g["n_truncated"] == o["n_truncated"]
    E = o["energy"]
    assert abs(g["energy"][0] - E) <= tolE * abs(E), (g["energy"][0], E)
    assert np.abs(g["atom_energy"] - o["atom_energy"]).max() <= 1e-11 * np.abs(o["atom_energy"]).max()
    rms = np.sqrt((o["forces"] ** 2).mean())
    assert np.abs(g["forces"] - o["forces"]).max() <= tolF * rms, (np.abs(g["forces"] - o["forces"]).max(), rms)
    vmax = np.abs(o["virial"]).max()
    assert np.abs(g["virial"] - o["virial"]).max() <= tolF * vmax


@pytest.mark.parametrize("idx", [0, 1])
def test_config_fp64_full_parity(idx):
    s = synth.config(idx)
    o = oracle.evaluate(s.coords, s.types, s.box, s.model)
    g = _gpu_eval(s)
    _check_fp64(g, o)


def test_coordinates_outside_box_and_type_map():
    s = synth.config(1)
    rng = np.random.default_rng(2)
    shift = rng.integers(-3, 4, size=(s.natoms, 3)) * 24.83
    s2 = synth.System(s.name, s.coords + shift, s.types, s.box, s.model, "fp64")
    o = oracle.evaluate(s.coords, s.types, s.box, s.model)
    g = _gpu_eval(s2)
    _check_fp64(g, o, tolE=2e-12, tolF=1e-9)     # coordinates differ by the rounding of the shift


def test_overflow_keeps_nearest_and_counts():
    s = synth.copper(5, 0.05, 77, sel=(100,))
    o = oracle.evaluate(s.coords, s.types, s.box, s.model)
    g = _gpu_eval(s)
    assert o["n_truncated"] == 500
    _check_fp64(g, o)


def test_ragged_small_and_padded_blocks():
    # water with generous capacities: many padded slots, ragged tile tails in both blocks
    s = synth.water(216, 18.7, 5, sel=(50, 100))
    o = oracle.evaluate(s.coords, s.types, s.box, s.model)
    g = _gpu_eval(s)
    _check_fp64(g, o)
