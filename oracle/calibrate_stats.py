"""Compute the per-centre-type normalisation statistics (avg, std) of a seeded configuration.

Run once (``python -m oracle.calibrate_stats``); the rounded numbers are frozen as constants in
paper_2005_00223_b200/synth.py (reading Q22).  Calls only oracle/ and the input generator.

Per centre type a, over all N_a * Nm slots (padded slots count as R~ = 0):
  avg_r = mean(s),  std_r = sqrt(mean(s^2) - avg_r^2),  avg_ang = 0,
  std_ang = sqrt(mean(R~_1^2 + R~_2^2 + R~_3^2) / 3).
"""
import numpy as np

from oracle import oracle
from paper_2005_00223_b200 import synth


def stats(coords, types, box, model):
    nl, dv, _ = oracle.nlist(coords, types, box, model.rc, model.sel)
    out = []
    for a in range(model.ntypes):
        rows = np.nonzero(types == a)[0]
        s_sum = s2_sum = ang2_sum = 0.0
        for i in rows:
            for k in np.nonzero(nl[i] >= 0)[0]:
                Rt, _ = oracle.env_row(dv[i, k], model.rc_smth, model.rc)
                s_sum += Rt[0]
                s2_sum += Rt[0] ** 2
                ang2_sum += Rt[1] ** 2 + Rt[2] ** 2 + Rt[3] ** 2
        nslots = len(rows) * model.nm
        avg = s_sum / nslots
        out.append((avg, np.sqrt(s2_sum / nslots - avg * avg), np.sqrt(ang2_sum / nslots / 3.0)))
    return out


if __name__ == "__main__":
    ideal = synth.copper(5, 0.0, 1)
    print("ideal FCC 5x5x5 (avg_r, std_r, std_ang):", stats(ideal.coords, ideal.types, ideal.box, ideal.model))
    w = synth.config(1)
    print("c1 water (per type):", stats(w.coords, w.types, w.box, w.model))
