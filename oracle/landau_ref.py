"""ctypes wrapper around the CPU oracle `liblandau_ref.so` (oracle/landau_ref.c).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs.  The product path (paper_2212_00663_b200) never imports
this module and shares no code with it.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "landau_ref.c"
_LIB = _HERE / "liblandau_ref.so"

_lib = None


def build(force: bool = False) -> Path:
    """Compile the oracle with gcc (-O2, OpenMP, no fast-math)."""
    if (not force and _LIB.exists()
            and _LIB.stat().st_mtime >= max(_SRC.stat().st_mtime, (_HERE / "landau_ref.h").stat().st_mtime)):
        return _LIB
    cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-fno-fast-math",
           "-Wall", "-Wextra", "-o", str(_LIB), str(_SRC), "-lm"]
    subprocess.run(cmd, check=True, cwd=str(_HERE))
    return _LIB


class StepInfo(C.Structure):
    _fields_ = [("iterations", C.c_int), ("residual", C.c_double), ("converged", C.c_int)]


def _load():
    global _lib
    if _lib is not None:
        return _lib
    build()
    lib = C.CDLL(str(_LIB))
    dp = C.POINTER(C.c_double)
    ip = C.POINTER(C.c_int32)
    lp = C.POINTER(C.c_int64)
    vp = C.c_void_p
    lib.landau_ref_gauss_hermite.argtypes = [C.c_int, dp, dp]
    lib.landau_ref_create.argtypes = [C.POINTER(vp), C.c_int, dp, dp, dp, C.c_int, C.c_double, dp]
    lib.landau_ref_destroy.argtypes = [vp]
    lib.landau_ref_destroy.restype = None
    lib.landau_ref_num_threads.restype = C.c_int
    lib.landau_ref_set_num_threads.argtypes = [C.c_int]
    lib.landau_ref_set_num_threads.restype = None
    lib.landau_ref_entropy_grad.argtypes = [vp, C.c_int64, dp, dp, ip, dp, dp]
    lib.landau_ref_entropy_grad_rows.argtypes = [vp, C.c_int64, dp, dp, ip, C.c_int64, lp, dp]
    lib.landau_ref_pair_field.argtypes = [vp, C.c_int64, dp, dp, ip, dp, dp]
    lib.landau_ref_pair_field_rows.argtypes = [vp, C.c_int64, dp, dp, ip, dp, C.c_int64, lp, dp]
    lib.landau_ref_eval_field.argtypes = [vp, C.c_int64, dp, dp, ip, dp]
    lib.landau_ref_set_markers.argtypes = [vp, C.c_int64, dp, dp, ip]
    lib.landau_ref_get_markers.argtypes = [vp, dp]
    lib.landau_ref_step.argtypes = [vp, C.c_double, C.c_double, C.c_int, C.POINTER(StepInfo)]
    lib.landau_ref_step_dg.argtypes = [vp, C.c_double, C.c_double, C.c_int, C.POINTER(StepInfo)]
    lib.landau_ref_moments.argtypes = [vp, dp, dp, dp, dp]
    lib.landau_ref_moments_ext.argtypes = [vp, dp, dp]
    _lib = lib
    return lib


def _d(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _i(a):
    return a.ctypes.data_as(C.POINTER(C.c_int32))


def _l(a):
    return a.ctypes.data_as(C.POINTER(C.c_int64))


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


class OracleError(RuntimeError):
    def __init__(self, code, where):
        super().__init__(f"landau_ref {where} failed with status {code}")
        self.code = code


def gauss_hermite(n: int):
    lib = _load()
    k = np.empty(n)
    a = np.empty(n)
    rc = lib.landau_ref_gauss_hermite(n, _d(k), _d(a))
    if rc:
        raise OracleError(rc, "gauss_hermite")
    return k, a


def num_threads() -> int:
    return int(_load().landau_ref_num_threads())


def set_num_threads(n: int) -> None:
    _load().landau_ref_set_num_threads(int(n))


class LandauRef:
    """Oracle context: species table + (optionally) held markers for stepping."""

    def __init__(self, mass, charge, eps, n_q: int = 4, nu0: float = 1.0, nu=None):
        lib = _load()
        self._lib = lib
        self.mass = _f64(mass)
        self.charge = _f64(charge)
        self.eps = _f64(eps)
        self.S = int(self.mass.shape[0])
        self.n_q = int(n_q)
        nu_arr = None if nu is None else _f64(nu)
        h = C.c_void_p()
        rc = lib.landau_ref_create(C.byref(h), self.S, _d(self.mass), _d(self.charge), _d(self.eps),
                                   self.n_q, float(nu0), None if nu_arr is None else _d(nu_arr))
        if rc:
            raise OracleError(rc, "create")
        self._h = h
        self.N = 0

    def close(self):
        if getattr(self, "_h", None):
            self._lib.landau_ref_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @staticmethod
    def _prep(v, w, sid):
        v = _f64(v)
        w = _f64(w)
        sid = np.ascontiguousarray(sid, dtype=np.int32)
        return v, w, sid, int(w.shape[0])

    def entropy_grad(self, v, w, sid, with_entropy: bool = False):
        v, w, sid, N = self._prep(v, w, sid)
        G = np.empty((N, 3))
        S = np.empty(self.S)
        rc = self._lib.landau_ref_entropy_grad(self._h, N, _d(v), _d(w), _i(sid), _d(G), _d(S))
        if rc:
            raise OracleError(rc, "entropy_grad")
        return (G, S) if with_entropy else G

    def entropy_grad_rows(self, v, w, sid, rows):
        v, w, sid, N = self._prep(v, w, sid)
        rows = np.ascontiguousarray(rows, dtype=np.int64)
        G = np.empty((rows.shape[0], 3))
        rc = self._lib.landau_ref_entropy_grad_rows(self._h, N, _d(v), _d(w), _i(sid), rows.shape[0], _l(rows), _d(G))
        if rc:
            raise OracleError(rc, "entropy_grad_rows")
        return G

    def pair_field(self, v, w, sid, G):
        v, w, sid, N = self._prep(v, w, sid)
        G = _f64(G)
        out = np.empty((N, 3))
        rc = self._lib.landau_ref_pair_field(self._h, N, _d(v), _d(w), _i(sid), _d(G), _d(out))
        if rc:
            raise OracleError(rc, "pair_field")
        return out

    def pair_field_rows(self, v, w, sid, G, rows):
        v, w, sid, N = self._prep(v, w, sid)
        G = _f64(G)
        rows = np.ascontiguousarray(rows, dtype=np.int64)
        out = np.empty((rows.shape[0], 3))
        rc = self._lib.landau_ref_pair_field_rows(self._h, N, _d(v), _d(w), _i(sid), _d(G), rows.shape[0], _l(rows), _d(out))
        if rc:
            raise OracleError(rc, "pair_field_rows")
        return out

    def eval_field(self, v, w, sid):
        v, w, sid, N = self._prep(v, w, sid)
        out = np.empty((N, 3))
        rc = self._lib.landau_ref_eval_field(self._h, N, _d(v), _d(w), _i(sid), _d(out))
        if rc:
            raise OracleError(rc, "eval_field")
        return out

    def set_markers(self, v, w, sid):
        v, w, sid, N = self._prep(v, w, sid)
        rc = self._lib.landau_ref_set_markers(self._h, N, _d(v), _d(w), _i(sid))
        if rc:
            raise OracleError(rc, "set_markers")
        self.N = N

    def get_markers(self):
        v = np.empty((self.N, 3))
        rc = self._lib.landau_ref_get_markers(self._h, _d(v))
        if rc:
            raise OracleError(rc, "get_markers")
        return v

    def step(self, dt, tol=1e-12, max_iter=50):
        """Returns (status, iterations, residual, converged); status 1 = not converged."""
        info = StepInfo()
        rc = self._lib.landau_ref_step(self._h, float(dt), float(tol), int(max_iter), C.byref(info))
        if rc < 0:
            raise OracleError(rc, "step")
        return rc, int(info.iterations), float(info.residual), bool(info.converged)

    def step_dg(self, dt, tol=1e-12, max_iter=50):
        """Discrete-gradient step, Eqs. (46)-(49) with Gonzalez' discrete gradient of S_eps (reading DG1)."""
        info = StepInfo()
        rc = self._lib.landau_ref_step_dg(self._h, float(dt), float(tol), int(max_iter), C.byref(info))
        if rc < 0:
            raise OracleError(rc, "step_dg")
        return rc, int(info.iterations), float(info.residual), bool(info.converged)

    def moments(self, with_entropy: bool = True):
        n = np.empty(self.S)
        P = np.empty((self.S, 3))
        K = np.empty(self.S)
        S = np.empty(self.S)
        rc = self._lib.landau_ref_moments(self._h, _d(n), _d(P), _d(K), _d(S) if with_entropy else None)
        if rc:
            raise OracleError(rc, "moments")
        return dict(n=n, P=P, K=K, S_eps=S if with_entropy else None)

    def moments_ext(self):
        stress = np.empty((self.S, 6))
        m4 = np.empty((self.S, 3))
        rc = self._lib.landau_ref_moments_ext(self._h, _d(stress), _d(m4))
        if rc:
            raise OracleError(rc, "moments_ext")
        return stress, m4
