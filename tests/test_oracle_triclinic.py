"""Pins of the oracle's general-cell (triclinic) neighbour search, reading N2t of DESIGN.md (-m "not gpu").

The paper takes the periodic images from LAMMPS' ghost region (Fig. 1(a)) and motivates arbitrary
multi-component systems; it gives no formula.  What fixes the answer without any implementation:
a rotated orthorhombic system is the same physical system; a re-chosen cell of the same lattice (a' = a + b) is the same
periodic system; a brute-force numpy enumeration of all images; energy finite differences; the strain derivative.
"""
import itertools

import numpy as np
import pytest

from oracle import oracle
from paper_2005_00223_b200 import synth


def _rot(seed):
    rng = np.random.default_rng(seed)
    q, r = np.linalg.qr(rng.standard_normal((3, 3)))
    q = q * np.sign(np.diag(r))
    if np.linalg.det(q) < 0:
        q[:, 0] = -q[:, 0]
    return q


def _sets(nl, sel):
    """per centre and per type block: sorted tuple of the listed neighbours (multiset; order-free comparison)"""
    off = np.concatenate([[0], np.cumsum(sel)])
    return [[tuple(sorted(int(v) for v in row[off[b]:off[b + 1]] if v >= 0)) for b in range(len(sel))] for row in nl]


def test_wrap_triclinic_lands_in_the_cell_and_moves_by_lattice_vectors():
    rng = np.random.default_rng(5)
    H = np.array([[7.0, 0.3, -0.2], [1.5, 6.0, 0.4], [-0.8, 1.1, 8.0]])
    for _ in range(50):
        x = rng.uniform(-40, 40, 3)
        xw = oracle.wrap_triclinic(H, x)
        f = xw @ np.linalg.inv(H)
        assert np.all(f > -1e-12) and np.all(f < 1 + 1e-12)
        n = (x - xw) @ np.linalg.inv(H)
        assert np.abs(n - np.round(n)).max() < 1e-12
    # a diagonal cell reproduces the per-axis wrap up to the rounding of x / L versus x * (1 / L)
    Hd = np.diag([5.0, 6.0, 7.0])
    x = np.array([17.3, -2.2, 7.5])
    assert np.allclose(oracle.wrap_triclinic(Hd, x), [oracle.wrap(x[k], Hd[k, k]) for k in range(3)], atol=1e-14)


@pytest.mark.parametrize("seed", [1, 2])
def test_rotated_orthorhombic_system_is_the_same_system(seed):
    """coordinates and cell rotated by a random rotation: the rotated cell is non-diagonal (general path, images of a box
    shorter than 2 rc included); E is invariant, forces and virial rotate, every list holds the same neighbours."""
    s = synth.small_fcc(2, 40 + seed, sigma=0.08, rc=4.2, rc_smth=1.2, sel=(48,), ntypes=2)     # L = 7.27 < 2 rc
    Q = _rot(seed)
    o = oracle.evaluate(s.coords, s.types, s.box, s.model)
    boxr = (s.box.reshape(3, 3) @ Q).reshape(9)
    r = oracle.evaluate(s.coords @ Q, s.types, boxr, s.model)
    assert np.abs(boxr.reshape(3, 3) - np.diag(np.diag(boxr.reshape(3, 3)))).max() > 0.5
    assert abs(r["energy"] - o["energy"]) <= 1e-12 * abs(o["energy"])
    assert np.abs(r["forces"] - o["forces"] @ Q).max() <= 1e-10 * np.abs(o["forces"]).max()
    V = o["virial"].reshape(3, 3)
    assert np.abs(r["virial"].reshape(3, 3) - Q.T @ V @ Q).max() <= 1e-10 * np.abs(V).max()
    assert _sets(r["nlist"], s.model.sel) == _sets(o["nlist"], s.model.sel)
    assert (o["nlist"] >= 0).sum(axis=1).min() >= 18      # two full FCC shells, images included (L < 2 rc)


def test_rechosen_cell_of_the_same_lattice_is_the_same_system():
    """a' = a + b, c' = c + a - b: another cell of the same lattice (det = 1 in lattice coordinates): same periodic system."""
    s = synth.small_fcc(3, 9, sigma=0.06, rc=4.5, rc_smth=1.0, sel=(40, 40), ntypes=2)          # L = 10.9 >= 2 rc
    H = s.box.reshape(3, 3)
    M = np.array([[1, 1, 0], [0, 1, 0], [1, -1, 1]])
    assert round(np.linalg.det(M)) == 1
    o = oracle.evaluate(s.coords, s.types, s.box, s.model)
    r = oracle.evaluate(s.coords, s.types, (M @ H).reshape(9), s.model)
    assert abs(r["energy"] - o["energy"]) <= 1e-12 * abs(o["energy"])
    assert np.abs(r["forces"] - o["forces"]).max() <= 1e-10 * np.abs(o["forces"]).max()
    assert np.abs(r["virial"] - o["virial"]).max() <= 1e-10 * np.abs(o["virial"]).max()
    assert _sets(r["nlist"], s.model.sel) == _sets(o["nlist"], s.model.sel)


def test_triclinic_list_against_numpy_brute_force():
    """a genuinely sheared cell with edges shorter than 2 rc: every (j, image) within rc by plain numpy enumeration"""
    rng = np.random.default_rng(11)
    H = np.array([[5.0, 0.0, 0.0], [2.1, 4.6, 0.0], [-1.3, 1.7, 5.2]])
    n = 10
    x = rng.random((n, 3)) @ H
    types = (np.arange(n) % 2).astype(np.int32)
    rc = 4.0
    sel = np.array([64, 64], dtype=np.int32)
    nl, dv, ntr = oracle.nlist(x, types, H.reshape(9), rc, sel)
    assert ntr == 0
    R = 3
    shifts = np.array(list(itertools.product(range(-R, R + 1), repeat=3))) @ H
    for i in range(n):
        want = {0: [], 1: []}
        for j in range(n):
            d = x[j] - x[i] + shifts
            r2 = (d ** 2).sum(1)
            k = np.count_nonzero(r2 < rc * rc) - (1 if j == i else 0)
            want[int(types[j])] += [j] * k
        got = _sets(nl[i:i + 1], sel)[0]
        assert got[0] == tuple(sorted(want[0])) and got[1] == tuple(sorted(want[1]))
        # the displacement vectors of the listed slots are images of x_j - x_i and sorted by distance within a block
        for b, o0 in ((0, 0), (1, 64)):
            m = nl[i, o0:o0 + 64] >= 0
            dd = dv[i, o0:o0 + 64][m]
            jj = nl[i, o0:o0 + 64][m]
            frac = (dd - (x[jj] - x[i])) @ np.linalg.inv(H)
            assert np.abs(frac - np.round(frac)).max() < 1e-9
            r = np.sqrt((dd ** 2).sum(1))
            assert np.all(np.diff(r) >= -1e-12) and np.all(r < rc)


def test_triclinic_forces_and_virial_by_finite_differences():
    rng = np.random.default_rng(3)
    H = np.array([[6.2, 0.0, 0.0], [1.9, 5.8, 0.0], [0.7, -1.4, 6.5]])
    n = 12
    x = rng.random((n, 3)) @ H
    types = (np.arange(n) % 2).astype(np.int32)
    m = synth.make_model(2, 4.0, 1.0, (40, 40), 77, [[0.1, 0, 0, 0]] * 2, [[0.2, 0.15, 0.15, 0.15]] * 2)
    o = oracle.evaluate(x, types, H.reshape(9), m)
    assert o["n_truncated"] == 0 and np.abs(o["forces"].sum(0)).max() < 1e-12
    h = 1e-5
    for (i, c) in ((0, 0), (3, 1), (7, 2), (11, 0)):
        xp, xm = x.copy(), x.copy()
        xp[i, c] += h; xm[i, c] -= h
        fd = -(oracle.energy(xp, types, H.reshape(9), m) - oracle.energy(xm, types, H.reshape(9), m)) / (2 * h)
        assert abs(fd - o["forces"][i, c]) <= 1e-7 * max(1.0, np.abs(o["forces"]).max())
    # Xi_ab = -dE/d(eps_ab): x -> x (1 + eps), H -> H (1 + eps)
    V = o["virial"].reshape(3, 3)
    for (a, b) in ((0, 0), (1, 2), (2, 0)):
        eps = np.zeros((3, 3)); eps[a, b] = h
        ep = oracle.energy(x @ (np.eye(3) + eps), types, (H @ (np.eye(3) + eps)).reshape(9), m)
        em = oracle.energy(x @ (np.eye(3) - eps), types, (H @ (np.eye(3) - eps)).reshape(9), m)
        assert abs(-(ep - em) / (2 * h) - V[a, b]) <= 1e-6 * np.abs(V).max()
