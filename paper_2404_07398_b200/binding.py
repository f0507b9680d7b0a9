"""Thin Python face of the C-ABI library (include/implicit_filter.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels of libimplicit_filter.so; PyTorch is used here for device
memory (fields, outputs, workspace) and streams.  There is no CPU path: if the library has not been built
(python -m paper_2404_07398_b200.build) or no CUDA device is present, calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libimplicit_filter.so")

IF_OK, IF_WNOTCONVERGED = 0, 1
IF_EINVAL, IF_EINDEX, IF_EDEGENERATE, IF_EORPHAN, IF_ENOMEM, IF_ECUDA, IF_EWORKSPACE, IF_EIO, IF_ELIMIT = -1, -2, -3, -4, -5, -6, -7, -8, -9
IF_FLAG_KEEP_CSR = 1
IF_FLAG_HIGHPASS = 2
IF_FLAG_MULTIGRID = 4
IF_FLAG_PAIRS = 8
IF_FLAG_VECTOR = 16
IF_FLAG_TRUE_RESIDUAL = 32

EXPORTS = ("if_prepare", "if_workspace_bytes", "if_filter", "if_spectrum", "if_spectrum_host", "if_apply", "if_mesh_info", "if_mesh_tile_info",
           "if_mesh_multigrid_info", "if_energy_noalloc",
           "if_mesh_export_csr", "if_mesh_export_perm", "if_save", "if_load", "if_destroy", "if_strerror", "if_launch_count")


class if_options(C.Structure):
    _fields_ = [("gamma", C.c_double), ("tol", C.c_double), ("max_iter", C.c_int), ("check_every", C.c_int),
                ("batch", C.c_int), ("sell_c", C.c_int), ("sell_sigma", C.c_int), ("sfc_kind", C.c_int),
                ("flags", C.c_int), ("solver", C.c_int), ("radius", C.c_double), ("mg_min_ell", C.c_double)]


class if_stats(C.Structure):
    _fields_ = [("iters", C.POINTER(C.c_int32)), ("rel_res", C.POINTER(C.c_double)),
                ("status", C.POINTER(C.c_int32)), ("seconds", C.c_double), ("batch_iters", C.c_int64),
                ("rhs_iters", C.c_int64), ("spmm_seconds", C.c_double), ("update_seconds", C.c_double),
                ("kernel_samples", C.c_int64), ("mg_kernel_seconds", C.c_double * 8), ("mg_samples", C.c_int64),
                ("mg_batch_iters", C.c_int64), ("true_res", C.POINTER(C.c_double))]


class ImplicitFilterError(RuntimeError):
    def __init__(self, code: int, what: str):
        super().__init__(f"{what}: {strerror(code)} ({code})")
        self.code = code


_lib = None


def load_library():
    """dlopen the in-tree library and declare its signatures.  Raises if it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_2404_07398_b200.build` "
                           "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    vp, i64, i32, dp = C.c_void_p, C.c_int64, C.c_int, C.POINTER(C.c_double)
    L.if_prepare.restype = i32
    L.if_prepare.argtypes = [vp, i32, i64, vp, i64, vp, C.POINTER(if_options), C.POINTER(vp)]
    L.if_workspace_bytes.restype = i32
    L.if_workspace_bytes.argtypes = [vp, i32, i32, C.POINTER(C.c_size_t)]
    L.if_filter.restype = i32
    L.if_filter.argtypes = [vp, vp, i32, vp, i32, i32, vp, vp, C.c_size_t, vp, C.POINTER(if_options),
                            C.POINTER(if_stats)]
    L.if_spectrum.restype = i32
    L.if_spectrum.argtypes = [vp, vp, i32, vp, i32, i32, vp, vp, vp, vp, C.c_size_t, vp, C.POINTER(if_options),
                              C.POINTER(if_stats)]
    L.if_spectrum_host.restype = i32
    L.if_spectrum_host.argtypes = L.if_spectrum.argtypes
    L.if_energy_noalloc.restype = i32
    L.if_energy_noalloc.argtypes = [vp, vp, i32, vp, vp]
    L.if_apply.restype = i32
    L.if_apply.argtypes = [vp, vp, i32, vp, i32, i32, vp, vp, C.c_size_t, vp, C.POINTER(if_options)]
    L.if_mesh_info.restype = i32
    L.if_mesh_info.argtypes = [vp, C.POINTER(i64), C.POINTER(i64), dp, dp, C.POINTER(i64)]
    L.if_mesh_tile_info.restype = i32
    L.if_mesh_tile_info.argtypes = [vp, C.POINTER(i64), C.POINTER(i64), C.POINTER(i64), C.POINTER(i64)]
    L.if_mesh_multigrid_info.restype = i32
    L.if_mesh_multigrid_info.argtypes = [vp, C.POINTER(C.c_int), vp, vp, vp, dp, vp]
    L.if_mesh_export_csr.restype = i32
    L.if_mesh_export_csr.argtypes = [vp, vp, vp, vp, vp]
    L.if_mesh_export_perm.restype = i32
    L.if_mesh_export_perm.argtypes = [vp, vp]
    L.if_save.restype = i32
    L.if_save.argtypes = [vp, C.c_char_p]
    L.if_load.restype = i32
    L.if_load.argtypes = [C.c_char_p, C.POINTER(vp)]
    L.if_destroy.restype = None
    L.if_destroy.argtypes = [vp]
    L.if_strerror.restype = C.c_char_p
    L.if_strerror.argtypes = [i32]
    L.if_launch_count.restype = i64
    L.if_launch_count.argtypes = []
    _lib = L
    return L


def strerror(code: int) -> str:
    return load_library().if_strerror(int(code)).decode()


def if_launch_count() -> int:
    return int(load_library().if_launch_count())


def _options(**kw) -> Optional[if_options]:
    kw = {k: v for k, v in kw.items() if v is not None}
    if not kw:
        return None
    o = if_options()
    for k, v in kw.items():
        if not hasattr(o, k):
            raise TypeError(f"unknown option {k!r}")
        setattr(o, k, v)
    return o


def _np_ptr(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


class Handle:
    """Owns an if_handle (device-resident prepared mesh) plus a side stream and a cached workspace."""

    def __init__(self, ptr: int, device):
        import torch
        self._ptr = C.c_void_p(ptr)
        self.device = device
        self.stream = torch.cuda.Stream(device=device)
        self._ws = None
        nv, nnz, slots = C.c_int64(), C.c_int64(), C.c_int64()
        ta, me = C.c_double(), C.c_double()
        load_library().if_mesh_info(self._ptr, C.byref(nv), C.byref(nnz), C.byref(ta), C.byref(me), C.byref(slots))
        self.n_vert, self.nnz, self.sell_slots = int(nv.value), int(nnz.value), int(slots.value)
        self.total_area, self.mean_edge = float(ta.value), float(me.value)
        nt, hr, hm, ut = C.c_int64(), C.c_int64(), C.c_int64(), C.c_int64()
        load_library().if_mesh_tile_info(self._ptr, C.byref(nt), C.byref(hr), C.byref(hm), C.byref(ut))
        self.n_tiles, self.halo_rows, self.halo_max, self.unstaged_tiles = (int(nt.value), int(hr.value),
                                                                            int(hm.value), int(ut.value))

    def close(self):
        if self._ptr is not None and self._ptr.value:
            load_library().if_destroy(self._ptr)
        self._ptr = None
        self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def workspace(self, order_n: int, batch: int = 0):
        import torch
        need = if_workspace_bytes(self, order_n, batch)
        if self._ws is None or self._ws.numel() < need:
            self._ws = None
            self._ws = torch.empty(need, dtype=torch.uint8, device=self.device)
        return self._ws


def if_prepare(coords, tri, period=None, **options) -> Handle:
    """Preparation phase: host arrays coords [V][dim] float64, tri [T][3] int32, period [dim] or None."""
    import torch
    L = load_library()
    if not torch.cuda.is_available():
        raise ImplicitFilterError(IF_ECUDA, "if_prepare (no CUDA device; there is no CPU fallback)")
    coords = np.ascontiguousarray(coords, dtype=np.float64)
    tri = np.ascontiguousarray(tri, dtype=np.int32)
    if coords.ndim != 2 or tri.ndim != 2 or tri.shape[1] != 3:
        raise ValueError("coords must be [V][dim], tri [T][3]")
    per = None if period is None else np.ascontiguousarray(period, dtype=np.float64)
    opt = _options(**options)
    out = C.c_void_p()
    device = torch.device("cuda", torch.cuda.current_device())
    torch.cuda.init()
    torch.zeros(1, device=device)      # make sure the primary context exists
    rc = L.if_prepare(_np_ptr(coords), coords.shape[1], coords.shape[0], _np_ptr(tri), tri.shape[0],
                      None if per is None else _np_ptr(per), None if opt is None else C.byref(opt), C.byref(out))
    if rc != IF_OK:
        raise ImplicitFilterError(rc, "if_prepare")
    return Handle(out.value, device)


def if_workspace_bytes(h: Handle, order_n: int, batch: int = 0) -> int:
    n = C.c_size_t()
    rc = load_library().if_workspace_bytes(h._ptr, int(order_n), int(batch), C.byref(n))
    if rc != IF_OK:
        raise ImplicitFilterError(rc, "if_workspace_bytes")
    return int(n.value)


def _device_fields(h: Handle, fields):
    import torch
    t = fields if isinstance(fields, torch.Tensor) else torch.from_numpy(np.ascontiguousarray(fields, dtype=np.float64))
    if t.dim() == 1:
        t = t[None, :]
    t = t.to(device=h.device, dtype=torch.float64).contiguous()
    if t.shape[1] != h.n_vert:
        raise ValueError(f"fields must be [F][{h.n_vert}]")
    return t


class _Stats:
    def __init__(self, n_rhs: int, shape):
        self.iters = np.zeros(n_rhs, dtype=np.int32)
        self.rel_res = np.zeros(n_rhs, dtype=np.float64)
        self.status = np.zeros(n_rhs, dtype=np.int32)
        self.shape = shape
        self.c = if_stats(self.iters.ctypes.data_as(C.POINTER(C.c_int32)),
                          self.rel_res.ctypes.data_as(C.POINTER(C.c_double)),
                          self.status.ctypes.data_as(C.POINTER(C.c_int32)), 0.0, 0, 0, 0.0, 0.0, 0)
        self.c.mg_samples = 0
        self.true_res = np.full(n_rhs, np.nan, dtype=np.float64)      # filled with IF_FLAG_TRUE_RESIDUAL
        self.c.true_res = self.true_res.ctypes.data_as(C.POINTER(C.c_double))

    def as_dict(self, rc: int):
        return {"iters": self.iters.reshape(self.shape), "rel_res": self.rel_res.reshape(self.shape),
                "status": self.status.reshape(self.shape), "true_res": self.true_res.reshape(self.shape),
                "seconds": float(self.c.seconds),
                "batch_iters": int(self.c.batch_iters), "rhs_iters": int(self.c.rhs_iters), "spmm_seconds": float(self.c.spmm_seconds),
                "update_seconds": float(self.c.update_seconds), "kernel_samples": int(self.c.kernel_samples),
                "mg_kernel_seconds": [float(v) for v in self.c.mg_kernel_seconds], "mg_samples": int(self.c.mg_samples),
                "mg_batch_iters": int(self.c.mg_batch_iters),
                "code": int(rc)}


def _run(h: Handle, what: str, call, stream):
    """Run `call(stream_ptr)` on the handle's side stream (ordered after the caller's current stream)."""
    import torch
    cur = torch.cuda.current_stream(h.device)
    st = h.stream if stream is None else stream
    st.wait_stream(cur)
    rc = call(C.c_void_p(st.cuda_stream))
    cur.wait_stream(st)
    if rc < 0:
        raise ImplicitFilterError(rc, what)
    return rc


def if_filter(h: Handle, fields, ells: Sequence[float], order_n: int, out=None, workspace=None, stream=None,
              **options):
    """Filtered fields [F][L][V] (torch.float64 on the device, caller's vertex order) and a stats dict."""
    import torch
    L = load_library()
    f = _device_fields(h, fields)
    el = np.ascontiguousarray(ells, dtype=np.float64)
    if out is None:
        out = torch.empty((f.shape[0], el.shape[0], h.n_vert), dtype=torch.float64, device=h.device)
    opt = _options(**options)
    ws = h.workspace(order_n, options.get("batch") or 0) if workspace is None else workspace
    st = _Stats(f.shape[0] * el.shape[0], (f.shape[0], el.shape[0]))
    rc = _run(h, "if_filter", lambda s: L.if_filter(
        h._ptr, C.c_void_p(f.data_ptr()), f.shape[0], _np_ptr(el), el.shape[0], int(order_n),
        C.c_void_p(out.data_ptr()), C.c_void_p(ws.data_ptr()), ws.numel(), s,
        None if opt is None else C.byref(opt), C.byref(st.c)), stream)
    return out, st.as_dict(rc)


def if_spectrum(h: Handle, fields, ells: Sequence[float], order_n: int, workspace=None, stream=None, **options):
    """dict(energy [F][L], k_mid [L-1], E [F][L-1], stats) -- host numpy arrays."""
    L = load_library()
    f = _device_fields(h, fields)
    el = np.ascontiguousarray(ells, dtype=np.float64)
    Fn, Ln = f.shape[0], el.shape[0]
    Fo = Fn // 2 if (options.get("flags") or 0) & IF_FLAG_PAIRS else Fn     # velocity pairs: one spectrum per (u, v)
    energy = np.zeros((Fo, Ln), dtype=np.float64)
    k_mid = np.zeros(max(Ln - 1, 0), dtype=np.float64)
    E = np.zeros((Fo, max(Ln - 1, 0)), dtype=np.float64)
    opt = _options(**options)
    ws = h.workspace(order_n, options.get("batch") or 0) if workspace is None else workspace
    st = _Stats(Fn * Ln, (Fn, Ln))
    rc = _run(h, "if_spectrum", lambda s: L.if_spectrum(
        h._ptr, C.c_void_p(f.data_ptr()), Fn, _np_ptr(el), Ln, int(order_n), _np_ptr(energy), _np_ptr(k_mid),
        _np_ptr(E), C.c_void_p(ws.data_ptr()), ws.numel(), s, None if opt is None else C.byref(opt),
        C.byref(st.c)), stream)
    return {"energy": energy, "k_mid": k_mid, "E": E, "stats": st.as_dict(rc)}


def if_spectrum_host(h: Handle, fields, ells: Sequence[float], order_n: int, workspace=None, stream=None, **options):
    """if_spectrum with the fields in HOST memory (numpy array or CPU torch tensor, ideally pinned): the C call copies
    them to the device itself.  Returns the same dict as if_spectrum."""
    import torch
    L = load_library()
    t = fields if isinstance(fields, torch.Tensor) else torch.from_numpy(np.ascontiguousarray(fields, dtype=np.float64))
    if t.dim() == 1:
        t = t[None, :]
    if t.device.type != "cpu" or t.dtype != torch.float64 or not t.is_contiguous() or t.shape[1] != h.n_vert:
        raise ValueError(f"fields must be a contiguous float64 HOST array [F][{h.n_vert}]")
    el = np.ascontiguousarray(ells, dtype=np.float64)
    Fn, Ln = t.shape[0], el.shape[0]
    Fo = Fn // 2 if (options.get("flags") or 0) & IF_FLAG_PAIRS else Fn     # velocity pairs: one spectrum per (u, v)
    energy = np.zeros((Fo, Ln), dtype=np.float64)
    k_mid = np.zeros(max(Ln - 1, 0), dtype=np.float64)
    E = np.zeros((Fo, max(Ln - 1, 0)), dtype=np.float64)
    opt = _options(**options)
    need = if_workspace_bytes(h, order_n, options.get("batch") or 0) + Fn * h.n_vert * 8
    if workspace is None:
        if h._ws is None or h._ws.numel() < need:
            h._ws = None
            h._ws = torch.empty(need, dtype=torch.uint8, device=h.device)
        workspace = h._ws
    st = _Stats(Fn * Ln, (Fn, Ln))
    rc = _run(h, "if_spectrum_host", lambda s: L.if_spectrum_host(
        h._ptr, C.c_void_p(t.data_ptr()), Fn, _np_ptr(el), Ln, int(order_n), _np_ptr(energy), _np_ptr(k_mid),
        _np_ptr(E), C.c_void_p(workspace.data_ptr()), workspace.numel(), s, None if opt is None else C.byref(opt),
        C.byref(st.c)), stream)
    return {"energy": energy, "k_mid": k_mid, "E": E, "stats": st.as_dict(rc)}


def if_energy_noalloc(h: Handle, fields, out=None, stream=None):
    """e_f = 1/2 sum_v A_v x_fv^2 / sum_v A_v for DEVICE fields [F][V] (torch.float64, caller's vertex order) into the
    DEVICE tensor `out` [F]: the entry point that allocates nothing (at most 32 fields per call; enqueued on the
    current torch stream, or `stream`, without synchronisation).  Pass `out` to keep the call itself allocation-free."""
    import torch
    if not isinstance(fields, torch.Tensor) or fields.device != h.device or fields.dtype != torch.float64 or \
            not fields.is_contiguous() or fields.dim() != 2 or fields.shape[1] != h.n_vert:
        raise ValueError(f"fields must be a contiguous float64 tensor [F][{h.n_vert}] on {h.device}")
    if out is None:
        out = torch.empty(fields.shape[0], dtype=torch.float64, device=h.device)
    st = torch.cuda.current_stream(h.device) if stream is None else stream
    rc = load_library().if_energy_noalloc(h._ptr, C.c_void_p(fields.data_ptr()), int(fields.shape[0]),
                                          C.c_void_p(out.data_ptr()), C.c_void_p(st.cuda_stream))
    if rc != IF_OK:
        raise ImplicitFilterError(rc, "if_energy_noalloc")
    return out


def if_apply(h: Handle, fields, ells: Sequence[float], order_n: int, out=None, workspace=None, stream=None,
             **options):
    """out[f][j] = (M + gamma l_j^(2n) S (M^-1 S)^(n-1)) fields[f]  -> torch.float64 [F][L][V] on the device."""
    import torch
    L = load_library()
    f = _device_fields(h, fields)
    el = np.ascontiguousarray(ells, dtype=np.float64)
    if out is None:
        out = torch.empty((f.shape[0], el.shape[0], h.n_vert), dtype=torch.float64, device=h.device)
    opt = _options(**options)
    ws = h.workspace(order_n, options.get("batch") or 0) if workspace is None else workspace
    _run(h, "if_apply", lambda s: L.if_apply(
        h._ptr, C.c_void_p(f.data_ptr()), f.shape[0], _np_ptr(el), el.shape[0], int(order_n),
        C.c_void_p(out.data_ptr()), C.c_void_p(ws.data_ptr()), ws.numel(), s,
        None if opt is None else C.byref(opt)), stream)
    return out


def if_mesh_export_csr(h: Handle):
    """(rowptr int64 [V+1], col int32 [nnz], val float64 [nnz], area float64 [V]) -- needs IF_FLAG_KEEP_CSR."""
    rowptr = np.empty(h.n_vert + 1, dtype=np.int64)
    col = np.empty(h.nnz, dtype=np.int32)
    val = np.empty(h.nnz, dtype=np.float64)
    area = np.empty(h.n_vert, dtype=np.float64)
    rc = load_library().if_mesh_export_csr(h._ptr, _np_ptr(rowptr), _np_ptr(col), _np_ptr(val), _np_ptr(area))
    if rc != IF_OK:
        raise ImplicitFilterError(rc, "if_mesh_export_csr")
    return rowptr, col, val, area


def if_mesh_multigrid_info(h: Handle) -> dict:
    """Levels of the multigrid hierarchy (rows, entries, prolongator entries), its build time and the sweep counts."""
    n = C.c_int(0)
    rows, nnz, pnnz = (np.zeros(12, dtype=np.int64) for _ in range(3))
    secs = C.c_double(0.0)
    sweeps = np.zeros(6, dtype=np.int32)
    rc = load_library().if_mesh_multigrid_info(h._ptr, C.byref(n), _np_ptr(rows), _np_ptr(nnz), _np_ptr(pnnz),
                                               C.byref(secs), _np_ptr(sweeps))
    if rc != IF_OK:
        raise ImplicitFilterError(rc, "if_mesh_multigrid_info")
    L = int(n.value)
    return {"levels": L, "rows": rows[:L].tolist(), "nnz": nnz[:L].tolist(), "p_nnz": pnnz[:L].tolist(),
            "build_seconds": float(secs.value), "sweeps": {1: sweeps[:3].tolist(), 2: sweeps[3:].tolist()}}


def if_mesh_export_perm(h: Handle) -> np.ndarray:
    perm = np.empty(h.n_vert, dtype=np.int32)
    rc = load_library().if_mesh_export_perm(h._ptr, _np_ptr(perm))
    if rc != IF_OK:
        raise ImplicitFilterError(rc, "if_mesh_export_perm")
    return perm


def if_save(h: Handle, path: str) -> None:
    """Write the prepared mesh to `path` (the auxiliary arrays are reusable)."""
    rc = load_library().if_save(h._ptr, os.fsencode(path))
    if rc != IF_OK:
        raise ImplicitFilterError(rc, "if_save")


def if_load(path: str) -> Handle:
    """A handle on the current CUDA device from a file written by if_save."""
    import torch
    if not torch.cuda.is_available():
        raise ImplicitFilterError(IF_ECUDA, "if_load (no CUDA device; there is no CPU fallback)")
    device = torch.device("cuda", torch.cuda.current_device())
    torch.zeros(1, device=device)
    out = C.c_void_p()
    rc = load_library().if_load(os.fsencode(path), C.byref(out))
    if rc != IF_OK:
        raise ImplicitFilterError(rc, "if_load")
    return Handle(out.value, device)


def if_destroy(h: Handle) -> None:
    h.close()
