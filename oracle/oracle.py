"""ctypes face of the CPU oracle (oracle/implicit_filter_oracle.c).

ORACLE -- test infrastructure, not product code.  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs import this.  It shares nothing with paper_2404_07398_b200/.
The arithmetic is all in the C file, which cites the paper passage each function follows; this
module only marshals numpy arrays.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Optional, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "implicit_filter_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None

GAMMA = 0.5        # PAPER.md:35 "Below we will take gamma = 1/2"
TOL = 1e-13        # BASELINE.json north_star: "fp64 CG to a relative residual of 1e-13"


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (no fast-math; OpenMP row loops only)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c11", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        vp, i64, i32, dbl = C.c_void_p, C.c_int64, C.c_int, C.c_double
        L.orc_build.restype = vp
        L.orc_build.argtypes = [vp, i32, i64, vp, i64, vp, C.POINTER(C.c_int)]
        L.orc_free.argtypes = [vp]
        L.orc_nv.restype = i64
        L.orc_nv.argtypes = [vp]
        L.orc_nnz.restype = i64
        L.orc_nnz.argtypes = [vp]
        L.orc_get_csr.argtypes = [vp, vp, vp, vp]
        L.orc_get_area.argtypes = [vp, vp]
        L.orc_apply_S.argtypes = [vp, vp, vp]
        L.orc_apply.argtypes = [vp, dbl, i32, dbl, vp, vp, vp]
        L.orc_solve.restype = i32
        L.orc_solve.argtypes = [vp, vp, dbl, i32, dbl, dbl, i64, vp, C.POINTER(i64), C.POINTER(dbl),
                                C.POINTER(dbl)]
        L.orc_energy.restype = dbl
        L.orc_energy.argtypes = [vp, vp]
        L.orc_spectrum.argtypes = [vp, vp, i32, vp, vp]
        L.orc_dense_solve.restype = i32
        L.orc_dense_solve.argtypes = [vp, vp, dbl, i32, dbl, vp]
        L.orc_threads.restype = i32
        L.orc_build_vector.restype = i32
        L.orc_build_vector.argtypes = [vp, vp, i32, vp, i64, vp, dbl]
        L.orc_get_vector_csr.argtypes = [vp, vp, vp]
        L.orc_apply_vector.argtypes = [vp, dbl, i32, dbl, vp, vp, vp, vp, vp]
        L.orc_solve_vector.restype = i32
        L.orc_solve_vector.argtypes = [vp, vp, vp, dbl, i32, dbl, dbl, i64, vp, vp, C.POINTER(i64), C.POINTER(dbl),
                                       C.POINTER(dbl)]
        _lib = L
    return _lib


def _p(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


def threads() -> int:
    return int(_load().orc_threads())


class OracleMesh:
    """S (CSR) and A_v assembled by the oracle from coordinates and triangles."""

    _ERR = {1: "bad triangle index", 2: "degenerate triangle", 3: "vertex in no triangle", 4: "out of memory"}

    def __init__(self, coords: np.ndarray, tri: np.ndarray, period: Optional[np.ndarray] = None):
        L = _load()
        coords = np.ascontiguousarray(coords, dtype=np.float64)
        tri = np.ascontiguousarray(tri, dtype=np.int32)
        per = None if period is None else np.ascontiguousarray(period, dtype=np.float64)
        err = C.c_int(0)
        self._h = L.orc_build(_p(coords), coords.shape[1], coords.shape[0], _p(tri), tri.shape[0],
                              None if per is None else _p(per), C.byref(err))
        if not self._h:
            raise ValueError("oracle: " + self._ERR.get(err.value, f"error {err.value}"))
        self.nv = int(L.orc_nv(self._h))
        self.nnz = int(L.orc_nnz(self._h))
        self._coords, self._tri, self._period = coords, tri, per          # kept for build_vector
        self._vector = False

    def __del__(self):
        if getattr(self, "_h", None) and _lib is not None:
            _lib.orc_free(self._h)
            self._h = None

    def csr(self) -> Tuple[np.ndarray, np.ndarray, np.ndarray]:
        rowptr = np.empty(self.nv + 1, dtype=np.int64)
        col = np.empty(self.nnz, dtype=np.int32)
        val = np.empty(self.nnz, dtype=np.float64)
        _load().orc_get_csr(self._h, _p(rowptr), _p(col), _p(val))
        return rowptr, col, val

    def area(self) -> np.ndarray:
        a = np.empty(self.nv, dtype=np.float64)
        _load().orc_get_area(self._h, _p(a))
        return a

    def apply_S(self, p: np.ndarray) -> np.ndarray:
        p = np.ascontiguousarray(p, dtype=np.float64)
        y = np.empty(self.nv, dtype=np.float64)
        _load().orc_apply_S(self._h, _p(p), _p(y))
        return y

    def apply(self, p: np.ndarray, ell: float, n: int, gamma: float = GAMMA) -> np.ndarray:
        """A_l p with A_l = M + gamma l^(2n) S (M^-1 S)^(n-1)."""
        p = np.ascontiguousarray(p, dtype=np.float64)
        y = np.empty(self.nv, dtype=np.float64)
        tmp = np.empty(self.nv, dtype=np.float64)
        _load().orc_apply(self._h, float(ell), int(n), float(gamma), _p(p), _p(y), _p(tmp))
        return y

    def solve(self, phi: np.ndarray, ell: float, n: int, gamma: float = GAMMA, tol: float = TOL,
              max_iter: int = 2_000_000):
        """Filtered field: Jacobi-PCG from x0 = phi.  Returns (x, info dict)."""
        phi = np.ascontiguousarray(phi, dtype=np.float64)
        x = np.empty(self.nv, dtype=np.float64)
        it = C.c_int64(0)
        rec = C.c_double(0.0)
        tru = C.c_double(0.0)
        st = _load().orc_solve(self._h, _p(phi), float(ell), int(n), float(gamma), float(tol), int(max_iter),
                               _p(x), C.byref(it), C.byref(rec), C.byref(tru))
        if st == 4:
            raise MemoryError("oracle: out of memory")
        return x, {"status": int(st), "iters": int(it.value), "rec_res": rec.value, "true_res": tru.value}

    def dense_solve(self, phi: np.ndarray, ell: float, n: int, gamma: float = GAMMA) -> np.ndarray:
        phi = np.ascontiguousarray(phi, dtype=np.float64)
        x = np.empty(self.nv, dtype=np.float64)
        st = _load().orc_dense_solve(self._h, _p(phi), float(ell), int(n), float(gamma), _p(x))
        if st != 0:
            raise RuntimeError(f"oracle dense solve failed ({st})")
        return x

    # ---- vector filter with metric terms
    def build_vector(self, radius: float = 0.0):
        """Assemble D~ and T (metric terms) on the pattern of S.  radius 0 => mean |x_v| (3-D meshes)."""
        if self._coords.shape[1] == 3 and radius == 0.0:
            radius = float(np.linalg.norm(self._coords, axis=1).mean())
        st = _load().orc_build_vector(self._h, _p(self._coords), self._coords.shape[1], _p(self._tri),
                                      self._tri.shape[0], None if self._period is None else _p(self._period),
                                      float(radius))
        if st != 0:
            raise MemoryError("oracle: out of memory")
        self._vector = True
        self.radius = radius

    def vector_csr(self):
        """(D~/l^2, T/l^2) values on the CSR pattern of csr()."""
        assert self._vector
        d = np.empty(self.nnz, dtype=np.float64)
        t = np.empty(self.nnz, dtype=np.float64)
        _load().orc_get_vector_csr(self._h, _p(d), _p(t))
        return d, t

    def apply_vector(self, pu, pv, ell: float, n: int, gamma: float = GAMMA):
        assert self._vector
        pu = np.ascontiguousarray(pu, dtype=np.float64)
        pv = np.ascontiguousarray(pv, dtype=np.float64)
        ou, ov = np.empty(self.nv), np.empty(self.nv)
        tmp = np.empty(4 * self.nv)
        _load().orc_apply_vector(self._h, float(ell), int(n), float(gamma), _p(pu), _p(pv), _p(ou), _p(ov), _p(tmp))
        return ou, ov

    def solve_vector(self, u, v, ell: float, n: int, gamma: float = GAMMA, tol: float = TOL, max_iter: int = 2_000_000):
        """Coarse-grained velocity (ubar, vbar) and an info dict."""
        assert self._vector
        u = np.ascontiguousarray(u, dtype=np.float64)
        v = np.ascontiguousarray(v, dtype=np.float64)
        xu, xv = np.empty(self.nv), np.empty(self.nv)
        it = C.c_int64(0)
        rec = C.c_double(0.0)
        tru = C.c_double(0.0)
        st = _load().orc_solve_vector(self._h, _p(u), _p(v), float(ell), int(n), float(gamma), float(tol), int(max_iter),
                                      _p(xu), _p(xv), C.byref(it), C.byref(rec), C.byref(tru))
        if st == 4:
            raise MemoryError("oracle: out of memory")
        return xu, xv, {"status": int(st), "iters": int(it.value), "rec_res": rec.value, "true_res": tru.value}

    def energy(self, x: np.ndarray) -> float:
        x = np.ascontiguousarray(x, dtype=np.float64)
        return float(_load().orc_energy(self._h, _p(x)))


def spectrum(ells: np.ndarray, e: np.ndarray):
    """(k_mid [L-1], E [L-1]) from cumulative energies e [L] at ascending scales ells [L]."""
    ells = np.ascontiguousarray(ells, dtype=np.float64)
    e = np.ascontiguousarray(e, dtype=np.float64)
    n = ells.shape[0]
    k_mid = np.empty(max(n - 1, 0), dtype=np.float64)
    E = np.empty(max(n - 1, 0), dtype=np.float64)
    _load().orc_spectrum(_p(ells), _p(e), n, _p(k_mid), _p(E))
    return k_mid, E


def filter_and_spectrum(mesh: OracleMesh, fields: np.ndarray, ells: np.ndarray, n: int, gamma: float = GAMMA,
                        tol: float = TOL, max_iter: int = 2_000_000):
    """All (field, scale) solves of one workload: filtered [F][L][V], energy [F][L], k_mid [L-1],
    E [F][L-1], infos [F][L]."""
    Fn, Ln = fields.shape[0], ells.shape[0]
    out = np.empty((Fn, Ln, mesh.nv), dtype=np.float64)
    en = np.empty((Fn, Ln), dtype=np.float64)
    infos = []
    for f in range(Fn):
        row = []
        for j in range(Ln):
            out[f, j], info = mesh.solve(fields[f], ells[j], n, gamma, tol, max_iter)
            en[f, j] = mesh.energy(out[f, j])
            row.append(info)
        infos.append(row)
    E = np.empty((Fn, max(Ln - 1, 0)), dtype=np.float64)
    k_mid = np.empty(max(Ln - 1, 0), dtype=np.float64)
    for f in range(Fn):
        k_mid, E[f] = spectrum(ells, en[f])
    return out, en, k_mid, E, infos
