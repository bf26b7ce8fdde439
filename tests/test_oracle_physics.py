"""Pins of the oracle's networks, energy, forces and virial (-m "not gpu").

Independent checks only: hand calculations, an independent numpy evaluation (library matmul / tanh, its own
minimum-image neighbour search), finite differences of the oracle's energy, and the invariances the paper
states (PAPER.md:49 "symmetry constraints", :51 continuity, :107 symmetries preserved, :109 permutation).
"""
import numpy as np
import pytest

from oracle import oracle
from paper_2005_00223_b200 import synth


# ------------------------------------------------------------------ nets: hand calculations
def test_embed_net_one_neuron_hand_calc():
    # widths (1, 2, 4): 1->1 would be "nout == nin" (identity skip); 1->2 and 2->4 are doubling layers
    W1, b1 = 0.7, -0.2
    W2 = np.array([[0.5, -1.5]]); b2 = np.array([0.1, 0.3])
    W3 = np.array([[1.0, 0.0, -0.5, 2.0], [0.25, -1.0, 0.5, 0.0]]); b3 = np.array([0.0, 0.1, -0.1, 0.2])
    net = np.concatenate([[W1], [b1], W2.ravel(), b2, W3.ravel(), b3])
    s = 0.37
    y1 = s + np.tanh(s * W1 + b1)                     # nout == nin == 1  -> x + tanh
    y2 = np.array([y1, y1]) + np.tanh(y1 * W2[0] + b2)
    G = np.concatenate([y2, y2]) + np.tanh(y2 @ W3 + b3)
    assert np.allclose(oracle.embed_net(net, (1, 2, 4), s), G, rtol=0, atol=1e-15)


def test_embed_net_zero_weights_doubling_is_copy():
    m = synth.config(0).model
    net = m.embed[:m.embed_net_size].copy()
    e = m.embed_net(0, 0)
    o = 50
    net[o:] = 0.0                                      # W2, b2, W3, b3 = 0  ->  G = (y1, y1, y1, y1)
    s = -0.4
    y1 = np.tanh(s * e["W1"][0] + e["b1"])
    assert np.allclose(oracle.embed_net(net, (25, 50, 100), s), np.tile(y1, 4), atol=1e-16)


def test_embed_and_fit_net_against_numpy_matmul():
    m = synth.config(1).model
    rng = np.random.default_rng(3)
    for (a, b) in ((0, 0), (0, 1), (1, 0), (1, 1)):
        e = m.embed_net(a, b)
        o = (a * 2 + b) * m.embed_net_size
        s = rng.standard_normal()
        y1 = np.tanh(np.array([s]) @ e["W1"] + e["b1"])
        y2 = np.concatenate([y1, y1]) + np.tanh(y1 @ e["W2"] + e["b2"])
        G = np.concatenate([y2, y2]) + np.tanh(y2 @ e["W3"] + e["b3"])
        assert np.allclose(oracle.embed_net(m.embed[o:o + m.embed_net_size], m.embed_widths, s), G, atol=1e-13)
    for a in (0, 1):
        f = m.fit_net(a)
        D = rng.standard_normal(1600) * 0.1
        h1 = np.tanh(D @ f["V1"] + f["c1"])
        h2 = h1 + np.tanh(h1 @ f["V2"] + f["c2"])
        h3 = h2 + np.tanh(h2 @ f["V3"] + f["c3"])
        E = h3 @ f["v4"] + f["c4"][0]
        o = a * m.fit_net_size
        assert abs(oracle.fit_net(m.fit[o:o + m.fit_net_size], 1600, m.fit_widths, D) - E) < 1e-12


def test_zero_weights_closed_form():
    s = synth.config(1)
    z = synth.make_model(2, 6.0, 0.5, (46, 92), 1, synth.WATER_AVG, synth.WATER_STD, zero=True)
    z.ebias[:] = [-3.5, -1.25]
    r = oracle.evaluate(s.coords[:300], s.types[:300], s.box, z)
    assert abs(r["energy"] - (100 * -3.5 + 200 * -1.25)) < 1e-10
    assert np.all(r["forces"] == 0) and np.all(r["virial"] == 0)


# ------------------------------------------------------------------ independent numpy evaluation of E
def numpy_energy(coords, types, L, m, want=False):
    """E by definition (N1..N7) with numpy; minimum image (needs L >= 2 rc); own sort."""
    N = len(coords)
    xw = coords - np.floor(coords / L) * L
    off = np.concatenate([[0], np.cumsum(m.sel)])
    Nm = int(off[-1])
    E = 0.0
    Ds = []
    for i in range(N):
        d = xw - xw[i]
        d -= L * np.round(d / L)
        r = np.sqrt((d ** 2).sum(1))
        Rhat = np.zeros((Nm, 4)); Gm = np.zeros((Nm, m.embed_widths[2]))
        a = types[i]
        for b in range(m.ntypes):
            idx = np.nonzero((r < m.rc) & (types == b) & (np.arange(N) != i))[0]
            idx = idx[np.argsort(r[idx], kind="stable")][:m.sel[b]]
            Rt = np.zeros((m.sel[b], 4))
            rr = r[idx]
            u = (rr - m.rc_smth) / (m.rc - m.rc_smth)
            w = np.where(rr < m.rc_smth, 1.0, u ** 3 * (-6 * u ** 2 + 15 * u - 10) + 1)
            Rt[:len(idx), 0] = w / rr
            Rt[:len(idx), 1:] = (w / rr ** 2)[:, None] * d[idx]
            Rh = (Rt - m.avg[a]) / m.std[a]
            e = m.embed_net(a, b)
            y1 = np.tanh(Rh[:, :1] @ e["W1"] + e["b1"])
            y2 = np.hstack([y1, y1]) + np.tanh(y1 @ e["W2"] + e["b2"])
            G = np.hstack([y2, y2]) + np.tanh(y2 @ e["W3"] + e["b3"])
            Rhat[off[b]:off[b + 1]] = Rh
            Gm[off[b]:off[b + 1]] = G
        A = Rhat.T @ Gm / Nm                              # [4, M1]
        D = (A.T @ A[:, :m.axis]).reshape(-1)             # [M1*M2], index m*M2 + a
        f = m.fit_net(a)
        h1 = np.tanh(D @ f["V1"] + f["c1"])
        h2 = h1 + np.tanh(h1 @ f["V2"] + f["c2"])
        h3 = h2 + np.tanh(h2 @ f["V3"] + f["c3"])
        E += h3 @ f["v4"] + f["c4"][0] + m.ebias[a]
        Ds.append(D)
    return (E, np.array(Ds)) if want else E


@pytest.mark.parametrize("ntypes", [1, 2])
def test_energy_against_independent_numpy(ntypes):
    s = synth.cluster(9, 21 + ntypes, ntypes=ntypes, sel=(6,) * ntypes)     # sel 6 < count -> truncation too
    r = oracle.evaluate(s.coords, s.types, s.box, s.model, want_descr=True)
    E, D = numpy_energy(s.coords, s.types, 40.0, s.model, want=True)
    assert np.allclose(r["descr"], D, rtol=1e-11, atol=1e-14)
    assert abs(r["energy"] - E) < 1e-11 * abs(E)


def test_energy_against_independent_numpy_water_subset():
    w = synth.config(1)
    E = numpy_energy(w.coords, w.types, 24.83, w.model)
    assert abs(oracle.energy(w.coords, w.types, w.box, w.model) - E) < 1e-11 * abs(E)


def test_descriptor_gram_block_is_symmetric_psd():
    s = synth.config(0)
    r = oracle.evaluate(s.coords, s.types, s.box, s.model, centers=np.array([0, 17, 401]), want_descr=True)
    for D in r["descr"]:
        B = D.reshape(100, 16)[:16]
        assert np.allclose(B, B.T, atol=1e-15)
        assert np.linalg.eigvalsh(B).min() > -1e-14


# ------------------------------------------------------------------ forces, virial: finite differences, invariances
def _fd_forces(s, atoms, h=1e-4):
    F = np.zeros((len(atoms), 3))
    for n, i in enumerate(atoms):
        for c in range(3):
            xp = s.coords.copy(); xp[i, c] += h
            xm = s.coords.copy(); xm[i, c] -= h
            F[n, c] = -(oracle.energy(xp, s.types, s.box, s.model) - oracle.energy(xm, s.types, s.box, s.model)) / (2 * h)
    return F


@pytest.mark.parametrize("which", ["cluster2", "fcc32_multi_image", "fcc108_two_types"])
def test_forces_equal_minus_grad_energy(which):
    if which == "cluster2":
        s = synth.cluster(8, 5, ntypes=2)
        atoms = range(8)
    elif which == "fcc32_multi_image":
        s = synth.small_fcc(2, 9, rc=5.0, rc_smth=1.5, sel=(96,))        # box 7.27 < 2 rc: several images
        atoms = [0, 13, 31]
    else:
        s = synth.small_fcc(3, 10, rc=5.0, rc_smth=1.0, sel=(40, 40), ntypes=2)
        atoms = [0, 50, 107]
    r = oracle.evaluate(s.coords, s.types, s.box, s.model)
    assert r["n_truncated"] == 0                                         # E is smooth only without overflow (Q14)
    F = _fd_forces(s, list(atoms))
    scale = np.abs(r["forces"]).max()
    assert np.abs(F - r["forces"][list(atoms)]).max() < 2e-7 * max(scale, 1e-3)
    assert np.abs(r["forces"].sum(0)).max() < 1e-12 * max(scale, 1.0) * s.natoms


def test_perfect_lattice_zero_force_isotropic_virial():
    s = synth.copper(5, 0.0, 3)
    r = oracle.evaluate(s.coords, s.types, s.box, s.model)
    assert np.abs(r["forces"]).max() < 1e-13
    V = r["virial"].reshape(3, 3)
    assert np.allclose(V, np.eye(3) * V[0, 0], atol=1e-10 * abs(V[0, 0]))
    assert np.allclose(r["atom_energy"], r["atom_energy"][0], atol=1e-13)


def test_translation_and_permutation_invariance():
    s = synth.small_fcc(3, 12, rc=5.0, rc_smth=1.0, sel=(40, 40), ntypes=2)
    r0 = oracle.evaluate(s.coords, s.types, s.box, s.model)
    r1 = oracle.evaluate(s.coords + np.array([1.234, -7.7, 25.01]), s.types, s.box, s.model)
    assert abs(r0["energy"] - r1["energy"]) < 1e-11 * abs(r0["energy"])
    assert np.abs(r0["forces"] - r1["forces"]).max() < 1e-11
    perm = np.random.default_rng(4).permutation(s.natoms)
    r2 = oracle.evaluate(s.coords[perm], s.types[perm], s.box, s.model)
    assert abs(r0["energy"] - r2["energy"]) < 1e-11 * abs(r0["energy"])
    assert np.abs(r0["forces"][perm] - r2["forces"]).max() < 1e-11
    assert np.abs(r0["atom_energy"][perm] - r2["atom_energy"]).max() < 1e-12


def test_rotation_invariance_and_covariance():
    s = synth.cluster(10, 8, ntypes=2)
    r0 = oracle.evaluate(s.coords, s.types, s.box, s.model)
    Q, _ = np.linalg.qr(np.random.default_rng(6).standard_normal((3, 3)))
    c = np.array([20.0, 20.0, 20.0])
    x1 = (s.coords - c) @ Q.T + c
    r1 = oracle.evaluate(x1, s.types, s.box, s.model)
    assert abs(r0["energy"] - r1["energy"]) < 1e-11 * abs(r0["energy"])
    assert np.abs(r0["forces"] @ Q.T - r1["forces"]).max() < 1e-11
    assert np.abs(Q @ r0["virial"].reshape(3, 3) @ Q.T - r1["virial"].reshape(3, 3)).max() < 1e-10
    # isolated cluster: no net torque, and virial = sum_i r_i (x) F_i
    x = s.coords - c
    assert np.abs(np.cross(x, r0["forces"]).sum(0)).max() < 1e-11
    assert np.abs(x.T @ r0["forces"] - r0["virial"].reshape(3, 3)).max() < 1e-11


def test_virial_equals_minus_strain_derivative():
    s = synth.small_fcc(3, 14, sigma=0.08, rc=5.0, rc_smth=1.0, sel=(90,))
    r = oracle.evaluate(s.coords, s.types, s.box, s.model)
    assert r["n_truncated"] == 0
    V = r["virial"].reshape(3, 3)
    assert np.abs(V - V.T).max() < 1e-11
    h = 1e-5
    for ax in range(3):
        def e(eps):
            sc = np.ones(3); sc[ax] += eps
            return oracle.energy(s.coords * sc, s.types, (s.box.reshape(3, 3) * sc).reshape(9), s.model)
        fd = -(e(h) - e(-h)) / (2 * h)
        assert abs(fd - V[ax, ax]) < 1e-6 * max(1.0, abs(V[ax, ax]))


def test_energy_continuous_across_rc_and_rc_smth():
    """Q4: padded rows are processed like a neighbour at r -> rc, so E does not jump when a slot fills."""
    m = synth.make_model(1, 6.0, 2.0, (4,), 31, [[0.3, 0, 0, 0]], [[0.2, 0.15, 0.15, 0.15]])
    types = np.zeros(3, dtype=np.int32)
    box = np.diag([40.0] * 3).reshape(9)

    def E(r):
        x = np.array([[20, 20, 20], [20 + r, 20, 20], [20, 23.1, 20.5]], dtype=np.float64)
        return oracle.energy(x, types, box, m)

    for edge in (6.0, 2.0):
        for h in (1e-3, 1e-4):
            jump = abs(E(edge + h) - E(edge - h))
            slope = abs(E(edge - h) - E(edge - 3 * h)) + 1e-300
            # C2 across the edge: the two-sided difference is no larger than a smooth function's
            assert jump < 3 * slope + 1e-13
    assert abs(E(6.0 + 1e-9) - E(6.0 - 1e-9)) < 1e-13
    # second derivative continuous: compare one-sided second differences
    h = 1e-3
    for edge in (6.0, 2.0):
        d2_in = (E(edge - 3 * h) - 2 * E(edge - 2 * h) + E(edge - h)) / h ** 2
        d2_out = (E(edge + 3 * h) - 2 * E(edge + 2 * h) + E(edge + h)) / h ** 2
        d2_far = (E(edge - 13 * h) - 2 * E(edge - 12 * h) + E(edge - 11 * h)) / h ** 2
        assert abs(d2_in - d2_out) < 10 * abs(d2_in - d2_far) + 1e-6


def test_dimer_force_along_bond():
    m = synth.make_model(1, 6.0, 1.0, (2,), 41, [[0.2, 0, 0, 0]], [[0.3, 0.2, 0.2, 0.2]])
    types = np.zeros(2, dtype=np.int32)
    box = np.diag([40.0] * 3).reshape(9)
    n = np.array([1.0, 2.0, -2.0]) / 3.0

    def ev(r):
        x = np.array([[20, 20, 20], [20, 20, 20] + r * n])
        return oracle.evaluate(x, types, box, m)

    r = 3.3
    out = ev(r)
    h = 1e-5
    dEdr = (ev(r + h)["energy"] - ev(r - h)["energy"]) / (2 * h)
    assert np.allclose(out["forces"][1], -dEdr * n, atol=1e-8)
    assert np.allclose(out["forces"][0], dEdr * n, atol=1e-8)
