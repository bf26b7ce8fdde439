"""Writes tests/golden/c4_full.npz: the CPU fp64 oracle (oracle/dp_oracle.c, nothing else) evaluated on EVERY atom of
BASELINE config 4 (copper, 1,048,576 atoms), reduced to what a test can compare without re-running the oracle
(about 10-20 minutes on 8-16 host cores):

  energy            total E (fp64)
  virial            Xi[9]
  rms_f             sqrt(mean F^2) over all 3 N force components (the RMS(F) of the north_star tolerance)
  subset            4,096 seeded atom indices;  forces_subset [4096,3], atom_energy_subset [4096]
  n_truncated       atoms with an over-full block
  nlist_group_sum   uint32 [N/16]: sum over 16 consecutive atoms (user order) of a 32-bit hash of the atom's formatted
                    neighbour row, see row_hash() below.  A GPU list that differs in any entry of any
                    row changes the hash of that row (the multipliers are odd, so a single changed entry always changes
                    the sum; several changed entries cancel only by 2^-32 chance).

Inputs come from the seeded generator paper_2005_00223_b200/synth.py (arrays only).  Nothing here touches the CUDA path.
Usage:  python tests/golden/make_full_size_golden.py [config_index=4]
"""
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

SUBSET = 4096
GROUP = 16


def row_hash(nl: np.ndarray) -> np.ndarray:
    """uint32 [rows]: sum_k (nl[i,k] + 2) * (2 k + 1) * 2654435761 mod 2^32 (entries are >= -1, so every term is > 0)."""
    k = np.arange(nl.shape[1], dtype=np.uint64)
    mult = ((2 * k + 1) * np.uint64(2654435761)) & np.uint64(0xFFFFFFFF)
    out = np.zeros(nl.shape[0], dtype=np.uint64)
    step = 1 << 16
    for r0 in range(0, nl.shape[0], step):
        v = (nl[r0:r0 + step].astype(np.int64) + 2).astype(np.uint64)
        out[r0:r0 + step] = (v * mult[None, :]).sum(axis=1) & np.uint64(0xFFFFFFFF)
    return out.astype(np.uint32)


def group_sums(h: np.ndarray) -> np.ndarray:
    n = (h.shape[0] + GROUP - 1) // GROUP * GROUP
    hp = np.zeros(n, dtype=np.uint64)
    hp[:h.shape[0]] = h
    return (hp.reshape(-1, GROUP).sum(axis=1) & np.uint64(0xFFFFFFFF)).astype(np.uint32)


def main():
    from oracle import oracle
    from paper_2005_00223_b200 import synth
    idx = int(sys.argv[1]) if len(sys.argv) > 1 else 4
    s = synth.config(idx)
    t0 = time.time()
    o = oracle.evaluate(s.coords, s.types, s.box, s.model)
    dt = time.time() - t0
    rng = np.random.default_rng(1000 + idx)
    subset = np.sort(rng.choice(s.natoms, size=min(SUBSET, s.natoms), replace=False)).astype(np.int64)
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), f"c{idx}_full.npz")
    np.savez_compressed(out, energy=np.float64(o["energy"]), virial=o["virial"],
                        rms_f=np.float64(np.sqrt((o["forces"] ** 2).mean())), subset=subset,
                        forces_subset=o["forces"][subset], atom_energy_subset=o["atom_energy"][subset],
                        n_truncated=np.int64(o["n_truncated"]), nlist_group_sum=group_sums(row_hash(o["nlist"])),
                        oracle_seconds=np.float64(dt), oracle_threads=np.int64(oracle.num_threads()))
    print(f"wrote {out}: N={s.natoms} E={o['energy']:.6f} oracle {dt:.1f} s on {oracle.num_threads()} threads")


if __name__ == "__main__":
    main()
