"""Pins of the CPU oracle against what the paper and the mathematics fix (-m "not gpu").

None of these compares the oracle with itself or with the CUDA path: closed forms (FCC shell census,
switch end points), invariants the paper states, finite differences, a
brute-force numpy evaluation written independently with library matmul/tanh, and hand calculations.
"""
import os

import numpy as np
import pytest

from oracle import oracle
from paper_2005_00223_b200 import synth

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


# ------------------------------------------------------------------ neighbour search / env matrix closed forms
def _read_shells():
    shells, sums = [], None
    for line in open(os.path.join(GOLDEN, "fcc_shells.txt")):
        if line.startswith("#") or not line.strip():
            continue
        tok = line.split()
        if tok[0] == "SUMS":
            sums = [float(t) for t in tok[1:]]
        else:
            shells.append((int(tok[0]), int(tok[1]), float(tok[2])))
    return shells, sums


def test_fcc_shell_census_and_env_values():
    """Ideal FCC: 176 neighbours in shells 12,6,24,12,24,8,48,6,36; per-shell s(r); avg/std closed form."""
    shells, sums = _read_shells()
    a, rc, rcs = 3.634, 8.0, 2.0
    s = synth.copper(5, 0.0, 1)
    nl, dv, ntr = oracle.nlist(s.coords, s.types, s.box, rc, s.model.sel)
    assert ntr == 0
    cnt = (nl >= 0).sum(1)
    assert np.all(cnt == 176)
    for i in (0, 137, 499):
        r = np.linalg.norm(dv[i, :176], axis=1)
        assert np.all(np.diff(r) >= -1e-9)            # sorted by distance (one type)
        pos = 0
        s_sum = s2_sum = ang2 = 0.0
        for n, mult, s_gold in shells:
            rr = r[pos:pos + mult]
            assert np.allclose(rr, a * np.sqrt(n / 2.0), atol=1e-9), (n, rr)
            for k in range(pos, pos + mult):
                Rt, _ = oracle.env_row(dv[i, k], rcs, rc)
                assert abs(Rt[0] - s_gold) < 2e-6
                s_sum += Rt[0]; s2_sum += Rt[0] ** 2; ang2 += (Rt[1:] ** 2).sum()
            pos += mult
        assert pos == 176
        assert abs(s_sum - sums[0]) < 2e-5 and abs(s2_sum - sums[1]) < 2e-5
        avg = s_sum / 256
        std = np.sqrt(s2_sum / 256 - avg ** 2)
        std_ang = np.sqrt(ang2 / 256 / 3)
        assert abs(avg - sums[2]) < 1e-6 and abs(std - sums[3]) < 1e-6 and abs(std_ang - sums[4]) < 1e-6
        assert abs((0 - avg) / std - sums[5]) < 1e-5
    # the recipe constants of the synthetic copper model are these closed-form numbers
    assert np.allclose(s.model.avg[0], [sums[2], 0, 0, 0], atol=1e-6)
    assert np.allclose(s.model.std[0], [sums[3], sums[4], sums[4], sums[4]], atol=1e-6)


def test_mean_neighbour_count_matches_density():
    """<count> = rho * 4/3 pi rc^3: 178.8 for copper; ~30.3 O + 60.5 H for water at 1.0 g/cm3."""
    s = synth.config(0)
    nl, _, _ = oracle.nlist(s.coords, s.types, s.box, s.model.rc, s.model.sel)
    assert abs((nl >= 0).sum(1).mean() - 4 / 3 * np.pi * 8.0 ** 3 * 4 / 3.634 ** 3) < 2.5
    w = synth.config(1)
    nl, _, _ = oracle.nlist(w.coords, w.types, w.box, w.model.rc, w.model.sel)
    rho_mol = 512 / 24.83 ** 3
    vol = 4 / 3 * np.pi * 6.0 ** 3
    assert abs((nl[:, :46] >= 0).sum(1).mean() - (rho_mol * vol - 1 / 3)) < 1.0
    assert abs((nl[:, 46:] >= 0).sum(1).mean() - (2 * rho_mol * vol - 2 / 3)) < 1.5


def test_switch_closed_form_values():
    rcs, rc = 2.0, 8.0
    assert oracle.switch(1.0, rcs, rc) == (1.0, 0.0)
    assert oracle.switch(rcs, rcs, rc)[0] == 1.0
    assert abs(oracle.switch(0.5 * (rcs + rc), rcs, rc)[0] - 0.5) < 1e-15
    assert oracle.switch(rc, rcs, rc) == (0.0, 0.0)
    assert oracle.switch(9.0, rcs, rc) == (0.0, 0.0)
    # monotone decreasing, derivative matches FD, C2 at both ends ("continuous to at least the 2nd order")
    rs = np.linspace(rcs, rc, 401)
    ws = np.array([oracle.switch(r, rcs, rc)[0] for r in rs])
    assert np.all(np.diff(ws) <= 1e-15)
    for r in (2.5, 4.0, 6.3, 7.9):
        h = 1e-6
        fd = (oracle.switch(r + h, rcs, rc)[0] - oracle.switch(r - h, rcs, rc)[0]) / (2 * h)
        assert abs(fd - oracle.switch(r, rcs, rc)[1]) < 1e-8
    for edge, inside in ((rcs, +1), (rc, -1)):
        h = 1e-3
        w0, d0 = oracle.switch(edge + inside * h, rcs, rc)
        target = 1.0 if edge == rcs else 0.0
        assert abs(w0 - target) < 20 * h ** 3        # w - w(edge) = O(h^3)
        assert abs(d0) < 20 * h ** 2                 # w' = O(h^2)  => w'' -> 0 as well
    # s = w/r is continuous at rc_smth (= 1/rc_smth) and at rc (= 0)
    Rt, _ = oracle.env_row([rcs * (1 - 1e-12), 0, 0], rcs, rc)
    assert abs(Rt[0] - 1 / rcs) < 1e-11
    Rt, _ = oracle.env_row([rc * (1 - 1e-9), 0, 0], rcs, rc)
    assert abs(Rt[0]) < 1e-15


def test_env_row_values_and_derivative():
    rng = np.random.default_rng(5)
    rcs, rc = 0.5, 6.0
    for _ in range(20):
        d = rng.standard_normal(3) * 2.0
        r = np.linalg.norm(d)
        if not (0.3 < r < rc):
            continue
        Rt, dRt = oracle.env_row(d, rcs, rc)
        w = oracle.switch(r, rcs, rc)[0]
        assert np.allclose(Rt, w / r * np.array([1, d[0] / r, d[1] / r, d[2] / r]), rtol=1e-14, atol=0)
        h = 1e-6
        for b in range(3):
            dp = d.copy(); dp[b] += h
            dm = d.copy(); dm[b] -= h
            fd = (oracle.env_row(dp, rcs, rc)[0] - oracle.env_row(dm, rcs, rc)[0]) / (2 * h)
            assert np.allclose(fd, dRt[:, b], atol=2e-8)


# ------------------------------------------------------------------ key / list structure
def test_key_order_is_lexicographic():
    rng = np.random.default_rng(11)
    n = 4000
    t = rng.integers(0, 4, n)
    r2 = rng.random(n) * 63.9
    r2[::7] = r2[3]                                       # equal distances -> tie broken by j
    j = rng.integers(0, 1 << 24, n)
    keys = np.array([oracle.key(int(a), float(b), int(c)) for a, b, c in zip(t, r2, j)], dtype=np.uint64)
    q = np.floor(r2 * 2.0 ** 29).astype(np.int64)
    lex = np.lexsort((j, q, t))
    assert np.array_equal(np.argsort(keys, kind="stable"), lex) or np.array_equal(keys[np.argsort(keys)], keys[lex])
    # fields decode back
    k = oracle.key(3, 17.25, 123456)
    assert k >> 60 == 3 and (k & ((1 << 24) - 1)) == 123456 and ((k >> 24) & ((1 << 36) - 1)) == int(17.25 * 2 ** 29)


def _check_rows(nl, dv, types, sel):
    off = np.concatenate([[0], np.cumsum(sel)])
    for i in range(nl.shape[0]):
        for b in range(len(sel)):
            blk = nl[i, off[b]:off[b + 1]]
            real = blk >= 0
            nreal = real.sum()
            assert np.all(real[:nreal]) and not np.any(real[nreal:])          # -1 only at the tail
            assert np.all(types[blk[:nreal]] == b)                            # block b holds type b only
            r2 = (dv[i, off[b]:off[b] + nreal] ** 2).sum(1)
            q = np.floor(r2 * 2.0 ** 29)
            key = q * 2.0 ** 24 + blk[:nreal]
            assert np.all(np.diff(key) > 0)                                   # strictly increasing keys


def test_nlist_structure_water_and_wrap():
    w = synth.config(1)
    sub = np.arange(0, w.natoms, 37)
    nl, dv, ntr = oracle.nlist(w.coords, w.types, w.box, w.model.rc, w.model.sel, centers=sub)
    _check_rows(nl, dv, w.types, w.model.sel)
    # atoms shifted by whole box vectors give the identical list (canonical wrap, N2)
    sh = w.coords + np.array([24.83, -2 * 24.83, 3 * 24.83])
    nl2, dv2, _ = oracle.nlist(sh, w.types, w.box, w.model.rc, w.model.sel, centers=sub)
    assert np.array_equal(nl, nl2) and np.allclose(dv, dv2, atol=1e-9)
    # brute force in numpy with minimum image (box >= 2 rc): same neighbour SETS
    L = 24.83
    xw = w.coords - np.floor(w.coords / L) * L
    for row, i in enumerate(sub[:12]):
        d = xw - xw[i]
        d -= L * np.round(d / L)
        r2 = (d ** 2).sum(1)
        mine = set(np.nonzero((r2 < 36.0) & (np.arange(w.natoms) != i))[0].tolist())
        assert set(nl[row][nl[row] >= 0].tolist()) == mine


def test_overflow_keeps_nearest():
    s = synth.copper(5, 0.05, 77, sel=(100,))
    full = synth.copper(5, 0.05, 77, sel=(256,))
    sub = np.arange(0, 500, 50)
    nl, dv, ntr = oracle.nlist(s.coords, s.types, s.box, 8.0, s.model.sel, centers=sub)
    nlf, dvf, _ = oracle.nlist(full.coords, full.types, full.box, 8.0, full.model.sel, centers=sub)
    assert ntr == len(sub)
    assert np.array_equal(nl, nlf[:, :100])                       # exactly the 100 nearest, same order
    r_kept = np.linalg.norm(dv[:, -1], axis=1)
    r_dropped = np.linalg.norm(dvf[:, 100], axis=1)
    assert np.all(r_kept <= r_dropped)


def test_small_box_multiple_images():
    """Box shorter than rc: an atom sees several images of the same neighbour and of itself."""
    x = np.array([[0.1, 0.2, 0.3], [1.7, 1.1, 0.9]])
    types = np.zeros(2, dtype=np.int32)
    box = np.diag([3.0, 3.0, 3.0]).reshape(9)
    rc = 3.5
    nl, dv, _ = oracle.nlist(x, types, box, rc, np.array([400], dtype=np.int32))
    # count lattice points by brute force in numpy
    g = np.arange(-3, 4)
    sh = np.stack(np.meshgrid(g, g, g, indexing="ij"), -1).reshape(-1, 3) * 3.0
    for i in range(2):
        n = 0
        for j in range(2):
            d = x[j] - x[i] + sh
            r = np.linalg.norm(d, axis=1)
            n += ((r < rc) & (r > 0)).sum()
        assert (nl[i] >= 0).sum() == n
