"""Seeded synthetic inputs for the DP (se_a) energy/force/virial path.

This module is the ONLY code shared by the CPU oracle (``oracle/``) and the CUDA
path (``paper_2005_00223_b200/csrc``).  It produces plain arrays -- coordinates,
types, box, a weight blob, model hyper-parameters -- and holds none of the
method's arithmetic (no switching function, no network evaluation, no
neighbour search).  The recipes follow BASELINE.json ``configs`` and SURVEY.md
section 8(d); the paper's own systems (section VI-A: water rc = 6 A,
copper rc = 8 A, fitting net (240,240,240)) and trained models are not
available, these seeded systems stand in for them.

Weight blob layout (fp64, row-major "in x out", y = x W + b as in PAPER.md:133):
  embed : T*T nets, index a*T + b (a = centre type, b = neighbour type), each
          W1[1*m0] b1[m0] W2[m0*m1] b2[m1] W3[m1*m2] b3[m2]
  fit   : T nets, each V1[(m2*axis)*f0] c1[f0] V2[f0*f1] c2[f1] V3[f1*f2] c3[f2]
          v4[f2] c4[1]
  ebias : [T]     avg : [T][4]     std : [T][4]   (per centre type)
"""
from __future__ import annotations

import dataclasses
import numpy as np

EMBED_WIDTHS = (25, 50, 100)
AXIS = 16
FIT_WIDTHS = (240, 240, 240)

# Per-centre-type normalisation constants of the synthetic models.  A trained DP
# model stores these numbers; here they are fixed constants of the recipe (see
# Q22).  Copper: the ideal-FCC closed-form values of
# SURVEY.md section 8(c) (a = 3.634, rc = 8, rc_smth = 2, capacity 256).  Water:
# rounded statistics of the seeded config-1 geometry, computed once with
# oracle/calibrate_stats.py and frozen here.
CU_AVG = (0.048849, 0.0, 0.0, 0.0)
CU_STD = (0.093189, 0.060746, 0.060746, 0.060746)
WATER_AVG = ((0.0511, 0.0, 0.0, 0.0), (0.0499, 0.0, 0.0, 0.0))
WATER_STD = ((0.1404, 0.0863, 0.0863, 0.0863), (0.1287, 0.0797, 0.0797, 0.0797))

# The paper's own network shape (section VI-A): embedding nets (32, 64, 128), fitting nets (240, 240, 240),
# neighbour capacities 512 (copper) and 144 (water: 48 O + 96 H).  Normalisation constants: the same statistics taken over
# the larger capacities (padded slots count as zero rows): copper from the ideal-FCC shell sums (sum s = 12.50524,
# sum s^2 = 2.83400 over 512 slots), water rescaled from the config-1 statistics (138 -> 144 slots).
PAPER_EMBED_WIDTHS = (32, 64, 128)
PAPER_CU_AVG = (0.024424, 0.0, 0.0, 0.0)
PAPER_CU_STD = (0.070275, 0.042954, 0.042954, 0.042954)
PAPER_WATER_AVG = ((0.04897, 0.0, 0.0, 0.0), (0.04782, 0.0, 0.0, 0.0))
PAPER_WATER_STD = ((0.13782, 0.08448, 0.08448, 0.08448), (0.12638, 0.07802, 0.07802, 0.07802))


@dataclasses.dataclass
class Model:
    ntypes: int
    rc: float
    rc_smth: float
    sel: np.ndarray          # int32 [T]
    embed_widths: tuple
    axis: int
    fit_widths: tuple
    embed: np.ndarray        # fp64 flat
    fit: np.ndarray          # fp64 flat
    ebias: np.ndarray        # fp64 [T]
    avg: np.ndarray          # fp64 [T,4]
    std: np.ndarray          # fp64 [T,4]

    @property
    def nm(self) -> int:
        return int(self.sel.sum())

    @property
    def embed_net_size(self) -> int:
        m0, m1, m2 = self.embed_widths
        return m0 + m0 + m0 * m1 + m1 + m1 * m2 + m2

    @property
    def fit_net_size(self) -> int:
        f0, f1, f2 = self.fit_widths
        d = self.embed_widths[2] * self.axis
        return d * f0 + f0 + f0 * f1 + f1 + f1 * f2 + f2 + f2 + 1

    def embed_net(self, a: int, b: int) -> dict:
        """Views of the (centre a, neighbour b) embedding net as named arrays."""
        m0, m1, m2 = self.embed_widths
        o = (a * self.ntypes + b) * self.embed_net_size
        e = self.embed
        out = {}
        out["W1"] = e[o:o + m0].reshape(1, m0); o += m0
        out["b1"] = e[o:o + m0]; o += m0
        out["W2"] = e[o:o + m0 * m1].reshape(m0, m1); o += m0 * m1
        out["b2"] = e[o:o + m1]; o += m1
        out["W3"] = e[o:o + m1 * m2].reshape(m1, m2); o += m1 * m2
        out["b3"] = e[o:o + m2]; o += m2
        return out

    def fit_net(self, a: int) -> dict:
        f0, f1, f2 = self.fit_widths
        d = self.embed_widths[2] * self.axis
        o = a * self.fit_net_size
        f = self.fit
        out = {}
        out["V1"] = f[o:o + d * f0].reshape(d, f0); o += d * f0
        out["c1"] = f[o:o + f0]; o += f0
        out["V2"] = f[o:o + f0 * f1].reshape(f0, f1); o += f0 * f1
        out["c2"] = f[o:o + f1]; o += f1
        out["V3"] = f[o:o + f1 * f2].reshape(f1, f2); o += f1 * f2
        out["c3"] = f[o:o + f2]; o += f2
        out["v4"] = f[o:o + f2]; o += f2
        out["c4"] = f[o:o + 1]; o += 1
        return out


@dataclasses.dataclass
class System:
    name: str
    coords: np.ndarray       # fp64 [N,3], Angstrom (may lie outside the box)
    types: np.ndarray        # int32 [N]
    box: np.ndarray          # fp64 [9] row-major, rows a, b, c (cubic here)
    model: Model
    precision: str           # "fp64" | "mix32" | "mix16"

    @property
    def natoms(self) -> int:
        return int(self.coords.shape[0])


def make_model(ntypes, rc, rc_smth, sel, seed, avg, std, ebias=-3.5,
               embed_widths=EMBED_WIDTHS, axis=AXIS, fit_widths=FIT_WIDTHS,
               bias_sigma=0.1, zero=False) -> Model:
    """W ~ N(0, 1/fan_in), biases ~ N(0, bias_sigma^2) (Q21), one seeded stream."""
    rng = np.random.default_rng(seed)
    m0, m1, m2 = embed_widths
    f0, f1, f2 = fit_widths
    d = m2 * axis

    def w(fan_in, fan_out):
        return rng.standard_normal(fan_in * fan_out) / np.sqrt(fan_in)

    def b(n):
        return bias_sigma * rng.standard_normal(n)

    emb = []
    for _a in range(ntypes):
        for _b in range(ntypes):
            emb += [w(1, m0), b(m0), w(m0, m1), b(m1), w(m1, m2), b(m2)]
    fit = []
    for _a in range(ntypes):
        fit += [w(d, f0), b(f0), w(f0, f1), b(f1), w(f1, f2), b(f2), w(f2, 1), b(1)]
    embed = np.ascontiguousarray(np.concatenate(emb))
    fitv = np.ascontiguousarray(np.concatenate(fit))
    if zero:
        embed[:] = 0.0
        fitv[:] = 0.0
    return Model(ntypes=ntypes, rc=float(rc), rc_smth=float(rc_smth),
                 sel=np.asarray(sel, dtype=np.int32), embed_widths=tuple(embed_widths),
                 axis=int(axis), fit_widths=tuple(fit_widths), embed=embed, fit=fitv,
                 ebias=np.full(ntypes, float(ebias)),
                 avg=np.asarray(avg, dtype=np.float64).reshape(ntypes, 4).copy(),
                 std=np.asarray(std, dtype=np.float64).reshape(ntypes, 4).copy())


# ----------------------------------------------------------------------------- copper
def fcc_positions(ncell: int, a: float = 3.634) -> np.ndarray:
    """Ideal FCC, conventional cell, basis (0,0,0),(0,.5,.5),(.5,0,.5),(.5,.5,0); cell-major order."""
    basis = np.array([[0, 0, 0], [0, .5, .5], [.5, 0, .5], [.5, .5, 0]], dtype=np.float64)
    g = np.arange(ncell, dtype=np.float64)
    cells = np.stack(np.meshgrid(g, g, g, indexing="ij"), axis=-1).reshape(-1, 1, 3)
    return ((cells + basis[None]) * a).reshape(-1, 3)


def copper(ncell: int, sigma: float, seed: int, shuffle: bool = False, a: float = 3.634,
           rc: float = 8.0, rc_smth: float = 2.0, sel=(256,), precision="fp64",
           name=None, embed_widths=EMBED_WIDTHS, avg=CU_AVG, std=CU_STD) -> System:
    rng = np.random.default_rng(seed)
    x = fcc_positions(ncell, a)
    x = x + sigma * rng.standard_normal(x.shape)
    if shuffle:
        x = x[rng.permutation(x.shape[0])]
    L = ncell * a
    box = np.diag([L, L, L]).reshape(9).astype(np.float64)
    model = make_model(1, rc, rc_smth, sel, seed + 1000, avg, std, embed_widths=embed_widths)
    return System(name or f"cu{x.shape[0]}", np.ascontiguousarray(x),
                  np.zeros(x.shape[0], dtype=np.int32), box, model, precision)


# ----------------------------------------------------------------------------- water
def _rsa_sites(n: int, L: float, dmin: float, rng) -> np.ndarray:
    """Random sequential addition of n points in a periodic cube, min-image distance >= dmin.

    Candidates are drawn in seeded batches and accepted with sequential semantics
    (a candidate is rejected iff it is closer than dmin to a point accepted earlier);
    scipy's periodic k-d tree only accelerates the distance queries.
    """
    from scipy.spatial import cKDTree
    pts = np.empty((0, 3), dtype=np.float64)
    while pts.shape[0] < n:
        batch = rng.random((min(65536, max(256, 32 * (n - pts.shape[0]))), 3)) * L
        if pts.shape[0]:
            dist, _ = cKDTree(pts, boxsize=L).query(batch, k=1, distance_upper_bound=dmin)
            batch = batch[~(dist < dmin)]
        if batch.shape[0] == 0:
            continue
        pairs = cKDTree(batch, boxsize=L).query_pairs(dmin, output_type="ndarray")
        ok = np.ones(batch.shape[0], dtype=bool)
        if pairs.shape[0]:
            # pairs (i<j): j is rejected if i was accepted; process in order of j then i
            lo = pairs.min(axis=1); hi = pairs.max(axis=1)
            order = np.lexsort((lo, hi))
            for i_, j_ in zip(lo[order], hi[order]):
                if ok[i_] and ok[j_]:
                    ok[j_] = False
        pts = np.concatenate([pts, batch[ok]])[:n]
    return np.ascontiguousarray(pts)


def _random_rotations(n: int, rng) -> np.ndarray:
    """Uniform random rotation matrices from unit quaternions (3 uniforms each)."""
    u = rng.random((n, 3))
    q = np.stack([np.sqrt(1 - u[:, 0]) * np.sin(2 * np.pi * u[:, 1]),
                  np.sqrt(1 - u[:, 0]) * np.cos(2 * np.pi * u[:, 1]),
                  np.sqrt(u[:, 0]) * np.sin(2 * np.pi * u[:, 2]),
                  np.sqrt(u[:, 0]) * np.cos(2 * np.pi * u[:, 2])], axis=1)
    x, y, z, w = q.T
    R = np.empty((n, 3, 3))
    R[:, 0, 0] = 1 - 2 * (y * y + z * z); R[:, 0, 1] = 2 * (x * y - z * w); R[:, 0, 2] = 2 * (x * z + y * w)
    R[:, 1, 0] = 2 * (x * y + z * w); R[:, 1, 1] = 1 - 2 * (x * x + z * z); R[:, 1, 2] = 2 * (y * z - x * w)
    R[:, 2, 0] = 2 * (x * z - y * w); R[:, 2, 1] = 2 * (y * z + x * w); R[:, 2, 2] = 1 - 2 * (x * x + y * y)
    return R


def water(nmol: int, L: float, seed: int, rc: float = 6.0, rc_smth: float = 0.5,
          sel=(46, 92), precision="fp64", name=None, embed_widths=EMBED_WIDTHS, avg=WATER_AVG, std=WATER_STD) -> System:
    rng = np.random.default_rng(seed)
    O = _rsa_sites(nmol, L, 2.5, rng)
    R = _random_rotations(nmol, rng)
    half = np.deg2rad(104.5) / 2
    h1 = 0.96 * np.array([np.sin(half), 0.0, np.cos(half)])
    h2 = 0.96 * np.array([-np.sin(half), 0.0, np.cos(half)])
    H1 = O + R @ h1
    H2 = O + R @ h2
    x = np.stack([O, H1, H2], axis=1).reshape(-1, 3)        # O,H,H per molecule
    types = np.tile(np.array([0, 1, 1], dtype=np.int32), nmol)
    box = np.diag([L, L, L]).reshape(9).astype(np.float64)
    model = make_model(2, rc, rc_smth, sel, seed + 1000, avg, std, embed_widths=embed_widths)
    return System(name or f"water{3 * nmol}", np.ascontiguousarray(x), types, box, model, precision)


# ----------------------------------------------------------------------------- the five configs
SEED0 = 20200500


def config(idx: int) -> System:
    """BASELINE.json configs[idx] (c0..c4)."""
    if idx == 0:
        return copper(5, 0.05, SEED0 + 0, name="c0_cu500", precision="fp64")
    if idx == 1:
        return water(512, 24.83, SEED0 + 1, name="c1_water1536", precision="fp64")
    if idx == 2:
        return copper(15, 0.05, SEED0 + 2, name="c2_cu13500", precision="fp64")
    if idx == 3:
        return water(36864, 97.4, SEED0 + 3, name="c3_water110592", precision="mix32")
    if idx == 4:
        return copper(64, 0.1, SEED0 + 4, shuffle=True, name="c4_cu1048576", precision="mix16")
    raise ValueError(idx)


# ----------------------------------------------------------------------------- the paper's network shape
def paper_copper(ncell: int, seed: int, sigma: float = 0.05, shuffle: bool = False, precision="fp64", name=None) -> System:
    """Copper with the paper's networks: embedding (32, 64, 128), capacity 512, rc 8 A."""
    return copper(ncell, sigma, seed, shuffle=shuffle, sel=(512,), precision=precision, name=name or f"paper_cu{4 * ncell ** 3}",
                  embed_widths=PAPER_EMBED_WIDTHS, avg=PAPER_CU_AVG, std=PAPER_CU_STD)


def paper_water(nmol: int, L: float, seed: int, precision="fp64", name=None) -> System:
    """Water with the paper's networks: embedding (32, 64, 128), capacity 144 = 48 O + 96 H, rc 6 A."""
    return water(nmol, L, seed, sel=(48, 96), precision=precision, name=name or f"paper_water{3 * nmol}",
                 embed_widths=PAPER_EMBED_WIDTHS, avg=PAPER_WATER_AVG, std=PAPER_WATER_STD)


def paper_config(name: str, precision="fp64") -> System:
    """Bench workloads at the paper's network shape: 'paper_cu' copper 32^3 cells = 131,072 atoms, 'paper_water' 36,864
    molecules = 110,592 atoms in the config-3 box (the paper's single-GPU runs: 4,860 Cu / 24,576 water atoms on a V100,
    PAPER.md Fig. 4; scaled to one B200)."""
    if name == "paper_cu":
        return paper_copper(32, SEED0 + 10, sigma=0.05, shuffle=True, precision=precision, name="paper_cu131072")
    if name == "paper_water":
        return paper_water(36864, 97.4, SEED0 + 11, precision=precision, name="paper_water110592")
    raise ValueError(name)


# ----------------------------------------------------------------------------- network-size study (Fig. 7)
SWEEP_WIDTHS = (64, 128, 256, 512)      # first embedding width W: last layer 2 W x 4 W = 128 x 256 ... 1024 x 2048


def wide_copper(ncell: int, W: int, seed: int, sigma: float = 0.05, shuffle: bool = False, sel=(512,), precision="mix16",
                name=None) -> System:
    """Copper (the system of Fig. 7) with embedding nets (W, 2 W, 4 W); capacity and statistics as paper_copper."""
    return copper(ncell, sigma, seed, shuffle=shuffle, sel=sel, precision=precision, name=name or f"wide{W}_cu{4 * ncell ** 3}",
                  embed_widths=(W, 2 * W, 4 * W), avg=PAPER_CU_AVG, std=PAPER_CU_STD)


def wide_water(nmol: int, L: float, W: int, seed: int, precision="mix16", name=None) -> System:
    """Two-type system with embedding nets (W, 2 W, 4 W): exercises the (centre, neighbour) type blocks of the wide path."""
    return water(nmol, L, seed, sel=(48, 96), precision=precision, name=name or f"wide{W}_water{3 * nmol}",
                 embed_widths=(W, 2 * W, 4 * W), avg=PAPER_WATER_AVG, std=PAPER_WATER_STD)


# ----------------------------------------------------------------------------- tiny systems for self-tests
def cluster(n: int, seed: int, ntypes: int = 1, L: float = 40.0, spread: float = 3.0,
            rc: float = 6.0, rc_smth: float = 1.0, sel=None, dmin: float = 1.2) -> System:
    """n atoms scattered in a ball of radius ~spread in a big box (isolated cluster)."""
    rng = np.random.default_rng(seed)
    pts = []
    while len(pts) < n:
        p = (rng.random(3) - 0.5) * 2 * spread
        if all(np.linalg.norm(p - q) >= dmin for q in pts):
            pts.append(p)
    x = np.array(pts) + L / 2
    types = (np.arange(n) % ntypes).astype(np.int32)
    rng.shuffle(types)
    sel = sel if sel is not None else tuple([max(4, n)] * ntypes)
    avg = [[0.1, 0, 0, 0]] * ntypes
    std = [[0.2, 0.15, 0.15, 0.15]] * ntypes
    model = make_model(ntypes, rc, rc_smth, sel, seed + 1000, avg, std)
    box = np.diag([L, L, L]).reshape(9).astype(np.float64)
    return System(f"cluster{n}", x, types, box, model, "fp64")


def small_fcc(ncell: int, seed: int, sigma: float = 0.05, a: float = 3.634, rc: float = 5.0,
              rc_smth: float = 1.5, sel=(64,), ntypes: int = 1, embed_widths=EMBED_WIDTHS) -> System:
    """Jittered FCC with a reduced cutoff (periodic, box may be < 2 rc: oracle-only)."""
    rng = np.random.default_rng(seed)
    x = fcc_positions(ncell, a)
    x = x + sigma * rng.standard_normal(x.shape)
    L = ncell * a
    n = x.shape[0]
    types = (rng.integers(0, ntypes, n)).astype(np.int32)
    sel = tuple(sel) if len(sel) == ntypes else tuple([sel[0]] * ntypes)
    avg = [[0.12, 0, 0, 0]] * ntypes
    std = [[0.15, 0.1, 0.1, 0.1]] * ntypes
    model = make_model(ntypes, rc, rc_smth, sel, seed + 1000, avg, std, embed_widths=embed_widths)
    box = np.diag([L, L, L]).reshape(9).astype(np.float64)
    return System(f"fcc{n}", np.ascontiguousarray(x), types, box, model, "fp64")


# ----------------------------------------------------------------------------- MD inputs
MASS_AMU = {"cu": (63.546,), "water": (15.999, 1.008)}     # per user type: copper; water O, H


def boltzmann_velocities(types: np.ndarray, masses, temperature: float, seed: int) -> np.ndarray:
    """Seeded velocities [N,3] in Angstrom/fs "randomly initialized subjected to the Boltzmann distribution"
    (330 K): each component ~ N(0, kB T / m), total momentum removed.  An input recipe only: the
    integrator arithmetic lives in csrc/md.cu and, independently, in oracle/md_oracle.py."""
    kb = 8.617333262e-5                                     # eV/K
    ev_per_amu_a2_fs2 = 1.0 / 9.648533216e-3                # 1 amu A^2/fs^2 in eV
    rng = np.random.Generator(np.random.PCG64(seed))
    m = np.asarray(masses, dtype=np.float64)[np.asarray(types)]
    v = rng.standard_normal((len(m), 3)) * np.sqrt(kb * temperature / (m * ev_per_amu_a2_fs2))[:, None]
    v -= (m[:, None] * v).sum(axis=0) / m.sum()
    return np.ascontiguousarray(v)
