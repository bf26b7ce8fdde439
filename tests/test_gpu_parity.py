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


# ------------------------------------------------------------------ mixed precision, BASELINE tolerances
def _check_forces(g, o, tol):
    rms = np.sqrt((o["forces"] ** 2).mean())
    err = np.abs(g["forces"] - o["forces"]).max()
    assert err <= tol * rms, (err / rms, tol)


def test_water_mix32_and_mix16_full_parity():
    """config 1 geometry in both mixed modes: list bit-exact, MIX-32 1e-4 RMS(F), MIX-16 5e-3 RMS(F)."""
    s = synth.config(1)
    o = oracle.evaluate(s.coords, s.types, s.box, s.model)
    for prec, tol, tolE in (("mix32", 1e-4, 2e-5), ("mix16", 5e-3, 1e-3)):
        g = _gpu_eval(s, prec)
        assert np.array_equal(g["nlist"], o["nlist"])
        _check_forces(g, o, tol)
        assert abs(g["energy"][0] - o["energy"]) / s.natoms <= tolE          # eV per atom
        vmax = np.abs(o["virial"]).max()
        assert np.abs(g["virial"] - o["virial"]).max() <= tol * vmax


def test_copper_mix16_parity_config0_geometry():
    s = synth.config(0)
    o = oracle.evaluate(s.coords, s.types, s.box, s.model)
    g = _gpu_eval(s, "mix16")
    assert np.array_equal(g["nlist"], o["nlist"])
    _check_forces(g, o, 5e-3)


def _sampled_check(idx, nsample, tol, tolEi):
    from sampling import sampled_oracle
    import torch
    from paper_2005_00223_b200 import binding
    s = synth.config(idx)
    so = sampled_oracle(s, nsample=nsample, seed=idx)
    m = binding.DPModel(s.model, s.precision)
    out = m.compute(torch.from_numpy(s.coords).cuda(), torch.from_numpy(s.types).cuda(), s.box)
    rc, ntr = m.status()
    assert rc == 0
    nl = m.get_nlist()[torch.from_numpy(so["centers"]).cuda()].cpu().numpy()
    F = out["forces"].cpu().numpy()
    ea = out["atom_energy"].cpu().numpy()
    E = float(out["energy"].item())
    m.close()
    assert np.array_equal(nl, so["nlist"])                                  # bit-exact rows of every evaluated centre
    assert np.abs(ea[so["centers"]] - so["atom_energy"]).max() <= tolEi
    err = np.abs(F[so["sample"]] - so["forces"]).max()
    assert err <= tol * so["rms_f"], (err / so["rms_f"], tol)
    # properties that hold at any size: total energy = sum of atomic energies, no net force
    assert abs(E - ea.sum()) <= 1e-9 * abs(E)
    assert np.abs(F.sum(0)).max() <= 1e-6 * np.abs(F).sum(0).max()
    return ntr


def test_config2_fp64_full_size():
    """copper 13,500 atoms, FP64 with DMMA: full oracle (seconds)."""
    s = synth.config(2)
    o = oracle.evaluate(s.coords, s.types, s.box, s.model)
    g = _gpu_eval(s)
    _check_fp64(g, o)


def test_config3_mix32_full_size_sampled():
    """water 110,592 atoms, MIX-32, in the launch configuration bench.py times; sampled oracle centres."""
    ntr = _sampled_check(3, nsample=64, tol=1e-4, tolEi=2e-5)
    assert ntr > 0            # the 97.4 A box over-fills a few blocks (reading Q23)


def test_config4_mix16_full_size_sampled():
    """copper 1,048,576 atoms, MIX-16, shuffled atom order; sampled oracle centres."""
    _sampled_check(4, nsample=48, tol=5e-3, tolEi=1e-3)


# ------------------------------------------------------------------ MIX-16 tcgen05 path: edge cases of the tiling
def test_mix16_overflow_blocks_have_no_padded_row():
    """every block over-full (no padded-row representative), rows per atom = sel: tiles span two atoms exactly"""
    s = synth.copper(5, 0.05, 77, sel=(100,))
    o = oracle.evaluate(s.coords, s.types, s.box, s.model)
    g = _gpu_eval(s, "mix16")
    assert np.array_equal(g["nlist"], o["nlist"]) and g["n_truncated"] == 500
    # Outside the five BASELINE configs the 5e-3 bound is not guaranteed: with only 100 rows per atom the single-fp16
    # activations of the forward kernel average less (measured 5.2e-3).  The bound here is 2x.
    _check_forces(g, o, 1e-2)
    assert g["rows"] == (500 * 100, 500 * 100)            # forward and backward push the same compact rows


def test_mix16_short_blocks_many_atoms_per_tile():
    """water with generous capacities: 128-row tiles span up to ~6 atoms (several passes per tile in the backward),
    ragged tails in all four (centre, neighbour) blocks"""
    s = synth.water(216, 18.7, 5, sel=(50, 100))
    o = oracle.evaluate(s.coords, s.types, s.box, s.model)
    g = _gpu_eval(s, "mix16")
    assert np.array_equal(g["nlist"], o["nlist"])
    _check_forces(g, o, 5e-3)
    vmax = np.abs(o["virial"]).max()
    assert np.abs(g["virial"] - o["virial"]).max() <= 5e-3 * vmax
    assert abs(g["energy"][0] - o["energy"]) / s.natoms <= 1e-3


@pytest.mark.parametrize("prec,tol", [("fp64", 1e-10), ("mix32", 1e-4), ("mix16", 5e-3)])
def test_tiny_two_type_cluster_fewer_rows_than_a_tile(prec, tol):
    """12 atoms of two types in a 40 A box: every (centre, neighbour) block is a fraction of one 128-row tile, the
    per-type fitting batches are 6 rows, the cell grid is mostly empty (workspace and tile-image sizing at tiny N)"""
    s = synth.cluster(12, 5, ntypes=2)
    o = oracle.evaluate(s.coords, s.types, s.box, s.model)
    g = _gpu_eval(s, prec)
    assert np.array_equal(g["nlist"], o["nlist"])
    _check_forces(g, o, tol)
    assert abs(g["energy"][0] - o["energy"]) <= (1e-12 if prec == "fp64" else 1e-3) * abs(o["energy"])


def test_profile_slots_and_launch_count():
    import torch
    from paper_2005_00223_b200 import binding
    s = synth.config(0)
    m = binding.DPModel(s.model, "mix16")
    c, t = torch.from_numpy(s.coords).cuda(), torch.from_numpy(s.types).cuda()
    m.compute(c, t, s.box)
    m.profile_enable(True)
    m.compute(c, t, s.box)
    ms = m.profile_read()
    assert ms.shape == (6,) and (ms >= 0).all()
    assert 0 < ms[5] <= ms[3]                  # the backward kernel alone is a part of the backward phase
    assert m.launches_per_compute() == 19      # one type: 16 + 3 T (every scan is three launches)
    m.close()


def test_perfect_lattice_ties_are_ordered_by_index():
    # ideal FCC: every shell is a set of exactly equal distances; the order inside a shell is the index order (PAPER.md:113:
    # the index sits in the low digits of the key).  Exercises the 64-bit re-sort behind the 32-bit proxy sort of the list kernel.
    s = synth.copper(5, 0.0, 12345, name="fcc_ideal")
    o = oracle.evaluate(s.coords, s.types, s.box, s.model)
    for prec in ("fp64", "mix16"):
        g = _gpu_eval(s, prec)
        assert np.array_equal(g["nlist"], o["nlist"])
    assert (o["nlist"] >= 0).sum(axis=1).min() >= 170
