"""ctypes front-end of the CPU fp64 oracle (oracle/dp_oracle.c).

TEST INFRASTRUCTURE -- only tests/, __graft_entry__.smoke() and the cpu_baseline /
``--impl reference`` legs of bench.py may import this.  It never imports the CUDA
package; models are duck-typed (attributes of paper_2005_00223_b200.synth.Model).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "dp_oracle.c")
_LIB = os.path.join(_HERE, "libdp_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """gcc -O2 -ffp-contract=off -fopenmp: no fused contractions the source does not spell out."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-std=c11",
               "-o", _LIB, _SRC, "-lm"]
        subprocess.check_call(cmd)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        dp, ip, lp = C.POINTER(C.c_double), C.POINTER(C.c_int), C.POINTER(C.c_long)
        L.oracle_num_threads.restype = C.c_int
        L.oracle_key.restype = C.c_uint64
        L.oracle_key.argtypes = [C.c_int, C.c_double, C.c_int]
        L.oracle_wrap.restype = C.c_double
        L.oracle_wrap.argtypes = [C.c_double, C.c_double]
        L.oracle_wrap_triclinic.restype = None
        L.oracle_wrap_triclinic.argtypes = [dp, dp, dp]
        L.oracle_switch.restype = C.c_double
        L.oracle_switch.argtypes = [C.c_double, C.c_double, C.c_double, dp]
        L.oracle_env_row.restype = None
        L.oracle_env_row.argtypes = [dp, C.c_double, C.c_double, dp, dp]
        L.oracle_embed_net.restype = None
        L.oracle_embed_net.argtypes = [dp, C.c_int, C.c_int, C.c_int, C.c_double, dp]
        L.oracle_fit_net.restype = C.c_double
        L.oracle_fit_net.argtypes = [dp, C.c_int, C.c_int, C.c_int, C.c_int, dp]
        L.oracle_nlist.restype = C.c_int
        L.oracle_nlist.argtypes = [C.c_long, dp, ip, dp, C.c_double, C.c_int, ip, C.c_long, lp, ip, dp, lp]
        L.oracle_eval_centers.restype = C.c_int
        L.oracle_eval_centers.argtypes = [C.c_int, ip] + [C.c_int] * 7 + [dp] * 5 + [C.c_double, C.c_double, ip,
                                          C.c_long, lp, ip, dp, dp, dp, dp, dp]
        L.oracle_assemble.restype = None
        L.oracle_assemble.argtypes = [C.c_long, lp, C.c_int, ip, dp, dp, dp, dp]
        _lib = L
    return _lib


def _d(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _i(a):
    return a.ctypes.data_as(C.POINTER(C.c_int))


def _l(a):
    return None if a is None else a.ctypes.data_as(C.POINTER(C.c_long))


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def key(type_j: int, r2: float, j: int) -> int:
    return int(lib().oracle_key(type_j, r2, j))


def wrap(x: float, L: float) -> float:
    return float(lib().oracle_wrap(x, L))


def wrap_triclinic(box, x) -> np.ndarray:
    box = np.ascontiguousarray(box, dtype=np.float64).reshape(9)
    x = np.ascontiguousarray(x, dtype=np.float64).reshape(3)
    out = np.zeros(3)
    lib().oracle_wrap_triclinic(_d(box), _d(x), _d(out))
    return out


def switch(r: float, rc_smth: float, rc: float):
    dw = C.c_double(0.0)
    w = lib().oracle_switch(r, rc_smth, rc, C.byref(dw))
    return float(w), float(dw.value)


def env_row(d, rc_smth: float, rc: float):
    d = np.ascontiguousarray(d, dtype=np.float64)
    Rt = np.zeros(4)
    dRt = np.zeros(12)
    lib().oracle_env_row(_d(d), rc_smth, rc, _d(Rt), _d(dRt))
    return Rt, dRt.reshape(4, 3)


def embed_net(net: np.ndarray, widths, s: float) -> np.ndarray:
    net = np.ascontiguousarray(net, dtype=np.float64)
    G = np.zeros(widths[2])
    lib().oracle_embed_net(_d(net), widths[0], widths[1], widths[2], float(s), _d(G))
    return G


def fit_net(net: np.ndarray, nd: int, widths, D: np.ndarray) -> float:
    net = np.ascontiguousarray(net, dtype=np.float64)
    D = np.ascontiguousarray(D, dtype=np.float64)
    return float(lib().oracle_fit_net(_d(net), nd, widths[0], widths[1], widths[2], _d(D)))


def nlist(coords, types, box, rc, sel, centers=None):
    """Formatted neighbour rows (user indices, -1 pad) + displacement vectors + #truncated centres."""
    coords = np.ascontiguousarray(coords, dtype=np.float64)
    types = np.ascontiguousarray(types, dtype=np.int32)
    box = np.ascontiguousarray(box, dtype=np.float64).reshape(9)
    sel = np.ascontiguousarray(sel, dtype=np.int32)
    N = coords.shape[0]
    cen = None if centers is None else np.ascontiguousarray(centers, dtype=np.int64)
    nc = N if cen is None else cen.shape[0]
    Nm = int(sel.sum())
    nl = np.empty((nc, Nm), dtype=np.int32)
    dv = np.empty((nc, Nm, 3), dtype=np.float64)
    ntr = C.c_long(0)
    rcode = lib().oracle_nlist(N, _d(coords), _i(types), _d(box), float(rc), int(sel.shape[0]), _i(sel), nc,
                               _l(cen), _i(nl), _d(dv), C.byref(ntr))
    if rcode != 0:
        raise ValueError(f"oracle_nlist failed with code {rcode}")
    return nl, dv, int(ntr.value)


def evaluate(coords, types, box, model, centers=None, want_descr=False):
    """Full DP evaluation (N1..N10).

    centers=None: every atom is a centre; returns energy, atom_energy [N], forces [N,3], virial [9].
    centers=array: only those centres are evaluated; ``forces``/``virial`` then hold the PARTIAL sums
    over the listed centres (complete for an atom i only if every atom within rc of i is listed).
    """
    coords = np.ascontiguousarray(coords, dtype=np.float64)
    types = np.ascontiguousarray(types, dtype=np.int32)
    box = np.ascontiguousarray(box, dtype=np.float64).reshape(9)
    N = coords.shape[0]
    sel = np.ascontiguousarray(model.sel, dtype=np.int32)
    Nm = int(sel.sum())
    nl, dv, ntr = nlist(coords, types, box, model.rc, sel, centers)
    cen = None if centers is None else np.ascontiguousarray(centers, dtype=np.int64)
    nc = nl.shape[0]
    m0, m1, m2 = model.embed_widths
    f0, f1, f2 = model.fit_widths
    ae = np.zeros(nc)
    gs = np.zeros((nc, Nm, 3))
    descr = np.zeros((nc, m2 * model.axis)) if want_descr else None
    amat = np.zeros((nc, 4, m2)) if want_descr else None
    emb = np.ascontiguousarray(model.embed, dtype=np.float64)
    fit = np.ascontiguousarray(model.fit, dtype=np.float64)
    eb = np.ascontiguousarray(model.ebias, dtype=np.float64)
    avg = np.ascontiguousarray(model.avg, dtype=np.float64)
    std = np.ascontiguousarray(model.std, dtype=np.float64)
    rcode = lib().oracle_eval_centers(int(model.ntypes), _i(sel), m0, m1, m2, int(model.axis), f0, f1, f2,
                                      _d(emb), _d(fit), _d(eb), _d(avg), _d(std), float(model.rc),
                                      float(model.rc_smth), _i(types), nc, _l(cen), _i(nl), _d(dv), _d(ae),
                                      _d(gs), None if descr is None else _d(descr),
                                      None if amat is None else _d(amat))
    if rcode != 0:
        raise ValueError(f"oracle_eval_centers failed with code {rcode}")
    F = np.zeros((N, 3))
    V = np.zeros(9)
    lib().oracle_assemble(nc, _l(cen), Nm, _i(nl), _d(dv), _d(gs), _d(F), _d(V))
    out = dict(energy=float(ae.sum()), atom_energy=ae, forces=F, virial=V, nlist=nl, dvec=dv, gslot=gs,
               n_truncated=ntr)
    if want_descr:
        out["descr"] = descr
        out["amat"] = amat
    return out


def energy(coords, types, box, model) -> float:
    return evaluate(coords, types, box, model)["energy"]
