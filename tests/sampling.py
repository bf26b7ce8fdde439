"""Sampled oracle parity for configurations too large for a full oracle evaluation.

Pick sample atoms; the oracle evaluates every centre within rc (+margin) of a sample atom, which makes the
assembled oracle force COMPLETE for the sample atoms (every slot gradient that touches them is included).
"""
import numpy as np
from scipy.spatial import cKDTree

from oracle import oracle


def sampled_oracle(s, nsample=32, seed=0, margin=1e-6):
    rng = np.random.default_rng(seed)
    L = float(s.box[0])
    assert s.box[0] == s.box[4] == s.box[8]
    xw = s.coords - np.floor(s.coords / L) * L
    xw = np.where(xw >= L, xw - L, xw)
    tree = cKDTree(xw, boxsize=L)
    sample = np.sort(rng.choice(s.natoms, size=min(nsample, s.natoms), replace=False))
    near = tree.query_ball_point(xw[sample], s.model.rc + margin)
    centers = np.unique(np.concatenate([np.asarray(n, dtype=np.int64) for n in near] + [sample]))
    o = oracle.evaluate(s.coords, s.types, s.box, s.model, centers=centers)
    return dict(sample=sample, centers=centers, forces=o["forces"][sample], atom_energy=o["atom_energy"],
                nlist=o["nlist"], rms_f=float(np.sqrt((o["forces"][sample] ** 2).mean())))
