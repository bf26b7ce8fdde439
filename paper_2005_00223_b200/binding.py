"""Thin Python binding of the C-ABI library (include/dp.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels of libdp_b200.so.  PyTorch is used for device
memory and streams.  There is no CPU fallback: a missing library or a missing GPU raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libdp_b200.so")
_lib = None

DP_FP64, DP_MIX32, DP_MIX16 = 0, 1, 2
PRECISIONS = {"fp64": DP_FP64, "mix32": DP_MIX32, "mix16": DP_MIX16}
EXPORTS = ["dp_create", "dp_workspace_bytes", "dp_compute", "dp_get_nlist", "dp_status",
           "dp_launches_per_compute", "dp_last_row_counts", "dp_profile_enable", "dp_profile_read", "dp_md_run",
           "dp_md_workspace_bytes", "dp_measure_peaks", "dp_last_cuda_error", "dp_destroy", "dp_strerror",
           "dp_scan_scratch_bytes", "dp_scan_exclusive", "dp_scan_exclusive_static"]
SCAN_STATIC_MAX = 16777216          # DP_SCAN_STATIC_MAX (include/dp.h)


class DPError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        msg = lib().dp_strerror(code).decode() if _lib is not None else str(code)
        super().__init__(f"{where}: {msg} ({code})")


class _Weights(C.Structure):
    _fields_ = [("ntypes", C.c_int), ("embed_widths", C.c_int * 3), ("axis", C.c_int), ("fit_widths", C.c_int * 3),
                ("embed", C.POINTER(C.c_double)), ("fit", C.POINTER(C.c_double)), ("ebias", C.POINTER(C.c_double)),
                ("avg", C.POINTER(C.c_double)), ("std", C.POINTER(C.c_double))]


def lib():
    """Load libdp_b200.so; fails loudly if it has not been built (python -m paper_2005_00223_b200.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2005_00223_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp, dp = C.c_void_p, C.POINTER(C.c_double)
        L.dp_strerror.restype = C.c_char_p
        L.dp_strerror.argtypes = [C.c_int]
        L.dp_create.restype = C.c_int
        L.dp_create.argtypes = [C.POINTER(vp), C.POINTER(_Weights), C.POINTER(C.c_int), C.c_int, C.c_double,
                                C.c_double, C.POINTER(C.c_int), C.c_int]
        L.dp_workspace_bytes.restype = C.c_size_t
        L.dp_workspace_bytes.argtypes = [vp, C.c_long, dp]
        L.dp_compute.restype = C.c_int
        L.dp_compute.argtypes = [vp, C.c_long, vp, vp, dp, vp, C.c_size_t, vp, vp, vp, vp, vp]
        L.dp_get_nlist.restype = C.c_int
        L.dp_get_nlist.argtypes = [vp, vp, vp]
        L.dp_status.restype = C.c_int
        L.dp_status.argtypes = [vp, C.POINTER(C.c_long)]
        L.dp_launches_per_compute.restype = C.c_int
        L.dp_launches_per_compute.argtypes = [vp]
        L.dp_last_row_counts.restype = C.c_int
        L.dp_last_row_counts.argtypes = [vp, C.POINTER(C.c_long), C.POINTER(C.c_long)]
        L.dp_profile_enable.restype = C.c_int
        L.dp_profile_enable.argtypes = [vp, C.c_int]
        L.dp_profile_read.restype = C.c_int
        L.dp_profile_read.argtypes = [vp, dp]
        L.dp_md_run.restype = C.c_int
        L.dp_md_run.argtypes = [vp, C.c_long, vp, vp, vp, dp, C.c_int, dp, C.c_double, C.c_int, C.c_double, C.c_int, vp,
                                C.c_size_t, vp, vp, vp, vp]
        L.dp_md_workspace_bytes.restype = C.c_size_t
        L.dp_md_workspace_bytes.argtypes = [vp, C.c_long, C.c_double, dp]
        L.dp_measure_peaks.restype = C.c_int
        L.dp_measure_peaks.argtypes = [dp, C.c_int, vp]
        L.dp_last_cuda_error.restype = C.c_char_p
        L.dp_last_cuda_error.argtypes = [vp, C.POINTER(C.c_int)]
        L.dp_destroy.restype = None
        L.dp_destroy.argtypes = [vp]
        L.dp_scan_scratch_bytes.restype = C.c_size_t
        L.dp_scan_scratch_bytes.argtypes = [C.c_int]
        L.dp_scan_exclusive.restype = C.c_int
        L.dp_scan_exclusive.argtypes = [C.c_int, vp, vp, vp, C.c_size_t, vp]
        L.dp_scan_exclusive_static.restype = C.c_int
        L.dp_scan_exclusive_static.argtypes = [C.c_int, vp, vp, vp]
        _lib = L
    return _lib


def _dptr(a: np.ndarray):
    return a.ctypes.data_as(C.POINTER(C.c_double))


class DPModel:
    """dp_create / dp_compute / dp_get_nlist / dp_status / dp_destroy with torch CUDA tensors."""

    def __init__(self, model, precision="fp64", type_map=None):
        L = lib()
        self._h = C.c_void_p(None)
        self.ntypes = int(model.ntypes)
        self.nm = int(np.sum(model.sel))
        w = _Weights()
        w.ntypes = self.ntypes
        w.embed_widths = (C.c_int * 3)(*model.embed_widths)
        w.axis = int(model.axis)
        w.fit_widths = (C.c_int * 3)(*model.fit_widths)
        keep = [np.ascontiguousarray(x, dtype=np.float64) for x in
                (model.embed, model.fit, model.ebias, model.avg, model.std)]
        w.embed, w.fit, w.ebias, w.avg, w.std = (_dptr(k) for k in keep)
        tm = np.ascontiguousarray(type_map if type_map is not None else np.arange(self.ntypes), dtype=np.int32)
        sel = np.ascontiguousarray(model.sel, dtype=np.int32)
        prec = PRECISIONS[precision] if isinstance(precision, str) else int(precision)
        rc = L.dp_create(C.byref(self._h), C.byref(w), tm.ctypes.data_as(C.POINTER(C.c_int)), int(tm.shape[0]),
                         float(model.rc), float(model.rc_smth), sel.ctypes.data_as(C.POINTER(C.c_int)), prec)
        if rc != 0:
            self._h = C.c_void_p(None)
            raise DPError(rc, "dp_create")
        self._ws = None
        self._n = 0

    def workspace_bytes(self, natoms: int, box=None) -> int:
        if box is None:
            return int(lib().dp_workspace_bytes(self._h, natoms, None))
        boxh = np.ascontiguousarray(np.asarray(box, dtype=np.float64).reshape(9))
        return int(lib().dp_workspace_bytes(self._h, natoms, _dptr(boxh)))

    def launches_per_compute(self) -> int:
        return int(lib().dp_launches_per_compute(self._h))

    def _workspace(self, natoms: int, device, box=None):
        import torch
        need = self.workspace_bytes(natoms, box)
        if need == 0:
            raise DPError(-2 if self.workspace_bytes(natoms) else -1, "dp_workspace_bytes")
        if self._ws is None or self._ws.numel() < need or self._ws.device != device:
            self._ws = torch.empty(need, dtype=torch.uint8, device=device)
        return self._ws

    def compute(self, coords, types, box, out=None, stream=None, want_virial=True, want_atom_energy=True):
        """coords [N,3] f64 cuda, types [N] i32 cuda, box 9 floats (host).  Enqueues only; returns output tensors."""
        import torch
        assert coords.is_cuda and types.is_cuda and coords.dtype == torch.float64 and types.dtype == torch.int32
        assert coords.is_contiguous() and types.is_contiguous()
        n = int(coords.shape[0])
        dev = coords.device
        ws = self._workspace(n, dev, box)
        if out is None:
            out = dict(energy=torch.empty(1, dtype=torch.float64, device=dev),
                       atom_energy=torch.empty(n, dtype=torch.float64, device=dev),
                       forces=torch.empty((n, 3), dtype=torch.float64, device=dev),
                       virial=torch.empty(9, dtype=torch.float64, device=dev))
        boxh = np.ascontiguousarray(np.asarray(box, dtype=np.float64).reshape(9))
        st = stream if stream is not None else torch.cuda.current_stream(dev)
        rc = lib().dp_compute(self._h, n, coords.data_ptr(), types.data_ptr(), _dptr(boxh), ws.data_ptr(),
                              ws.numel(), st.cuda_stream, out["energy"].data_ptr(),
                              out["atom_energy"].data_ptr() if want_atom_energy else None,
                              out["forces"].data_ptr(), out["virial"].data_ptr() if want_virial else None)
        if rc != 0:
            where = "dp_compute"
            if rc == -5:
                step = C.c_int(0)
                where += f" [{lib().dp_last_cuda_error(self._h, C.byref(step)).decode()}, call {step.value}]"
            raise DPError(rc, where)
        self._n = n
        return out

    def md_run(self, coords, vel, types, masses, box, dt_fs, nsteps, skin=0.0, rebuild_every=0, stream=None,
               want_virial=True):
        """Velocity-Verlet loop (dp_md_run): coords, vel [N,3] f64 cuda are advanced IN PLACE by nsteps steps of dt_fs;
        masses: amu per user type; skin > 0 and rebuild_every > 1: buffered neighbour list.
        Enqueues only; returns forces [N,3], thermo [nsteps+1,4] (E_pot eV, E_kin eV, T K, P bar), virial."""
        import torch
        for x in (coords, vel):
            assert x.is_cuda and x.dtype == torch.float64 and x.is_contiguous()
        assert types.is_cuda and types.dtype == torch.int32 and types.is_contiguous()
        n = int(coords.shape[0])
        dev = coords.device
        buffered = skin > 0.0 and rebuild_every > 1
        boxh = np.ascontiguousarray(np.asarray(box, dtype=np.float64).reshape(9))
        need = int(lib().dp_md_workspace_bytes(self._h, n, float(skin) if buffered else 0.0, _dptr(boxh)))
        if need == 0:
            raise DPError(-1, "dp_md_workspace_bytes")
        if self._ws is None or self._ws.numel() < need or self._ws.device != dev:
            self._ws = torch.empty(need, dtype=torch.uint8, device=dev)
        ws = self._ws
        out = dict(forces=torch.empty((n, 3), dtype=torch.float64, device=dev),
                   thermo=torch.empty((int(nsteps) + 1, 4), dtype=torch.float64, device=dev),
                   virial=torch.empty(9, dtype=torch.float64, device=dev))
        boxh = np.ascontiguousarray(np.asarray(box, dtype=np.float64).reshape(9))
        mh = np.ascontiguousarray(masses, dtype=np.float64)
        st = stream if stream is not None else torch.cuda.current_stream(dev)
        rc = lib().dp_md_run(self._h, n, coords.data_ptr(), vel.data_ptr(), types.data_ptr(), _dptr(mh), int(mh.shape[0]),
                             _dptr(boxh), float(dt_fs), int(nsteps), float(skin), int(rebuild_every), ws.data_ptr(), ws.numel(),
                             st.cuda_stream,
                             out["forces"].data_ptr(), out["thermo"].data_ptr(),
                             out["virial"].data_ptr() if want_virial else None)
        if rc != 0:
            raise DPError(rc, "dp_md_run")
        self._n = n
        return out

    def get_nlist(self, stream=None):
        import torch
        dev = self._ws.device
        nl = torch.empty((self._n, self.nm), dtype=torch.int32, device=dev)
        st = stream if stream is not None else torch.cuda.current_stream(dev)
        rc = lib().dp_get_nlist(self._h, nl.data_ptr(), st.cuda_stream)
        if rc != 0:
            raise DPError(rc, "dp_get_nlist")
        return nl

    def status(self):
        nt = C.c_long(0)
        rc = lib().dp_status(self._h, C.byref(nt))
        return rc, int(nt.value)

    def last_row_counts(self):
        a, b = C.c_long(0), C.c_long(0)
        rc = lib().dp_last_row_counts(self._h, C.byref(a), C.byref(b))
        if rc != 0:
            raise DPError(rc, "dp_last_row_counts")
        return int(a.value), int(b.value)

    def profile_enable(self, on=True):
        rc = lib().dp_profile_enable(self._h, 1 if on else 0)
        if rc != 0:
            raise DPError(rc, "dp_profile_enable")

    def profile_read(self):
        """Per-phase milliseconds of the last compute: nlist, embed_fwd, fit, embed_bwd, finalize."""
        ms = np.zeros(6)
        rc = lib().dp_profile_read(self._h, _dptr(ms))
        if rc != 0:
            raise DPError(rc, "dp_profile_read")
        return ms

    def close(self):
        if self._h:
            lib().dp_destroy(self._h)
            self._h = C.c_void_p(None)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def measure_peaks(stream=None) -> dict:
    """dp_measure_peaks on the current device: measured DFMA / DMMA / FFMA / tanh.approx / mma.sync rates."""
    import torch
    out = np.zeros(6)
    st = stream if stream is not None else torch.cuda.current_stream()
    rc = lib().dp_measure_peaks(_dptr(out), 6, st.cuda_stream)
    if rc != 0:
        raise DPError(rc, "dp_measure_peaks")
    return dict(dfma_tflops=out[0], dmma_tflops=out[1], ffma_tflops=out[2], tanh_tera_per_s=out[3],
                hmma_sync_tflops=out[4], sms=int(out[5]))


def scan_exclusive(cnt, out, scratch, stream=None) -> None:
    """dp_scan_exclusive: out[0..n] = exclusive prefix sums of cnt[0..n) (int32 CUDA tensors), caller-owned scratch tensor."""
    import torch
    st = stream if stream is not None else torch.cuda.current_stream()
    rc = lib().dp_scan_exclusive(int(cnt.numel()), cnt.data_ptr(), out.data_ptr(), scratch.data_ptr(),
                                 scratch.numel() * scratch.element_size(), st.cuda_stream)
    if rc != 0:
        raise DPError(rc, "dp_scan_exclusive")


def scan_exclusive_static(cnt, out, stream=None) -> None:
    """dp_scan_exclusive_static: the same result with the scratch in a static device array of the library: no allocation,
    n <= SCAN_STATIC_MAX; calls that overlap on the GPU race on that array (include/dp.h)."""
    import torch
    st = stream if stream is not None else torch.cuda.current_stream()
    rc = lib().dp_scan_exclusive_static(int(cnt.numel()), cnt.data_ptr(), out.data_ptr(), st.cuda_stream)
    if rc != 0:
        raise DPError(rc, "dp_scan_exclusive_static")


def compute_host(model_handle: DPModel, coords_np, types_np, box, device="cuda:0"):
    """End-to-end convenience call with HOST buffers: H2D copy, dp_compute, D2H copy, status check."""
    import torch
    c = torch.from_numpy(np.ascontiguousarray(coords_np, dtype=np.float64)).to(device)
    t = torch.from_numpy(np.ascontiguousarray(types_np, dtype=np.int32)).to(device)
    out = model_handle.compute(c, t, box)
    rc, ntr = model_handle.status()
    if rc != 0:
        raise DPError(rc, "dp_status")
    res = {k: v.cpu().numpy() for k, v in out.items()}
    res["energy"] = float(res["energy"][0])
    res["n_truncated"] = ntr
    return res
