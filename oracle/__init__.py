"""CPU ORACLE binding (ctypes over oracle/wl_oracle.cpp).  TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl
reference`` legs may import this package.  It imports nothing from ``paper_2304_08159_b200``'s
CUDA binding and shares no code with it.  Arrays are NumPy, shapes as in
``paper_2304_08159_b200/synth.py``: cell field ``(N_{n-1},…,N_0)``, face field ``(n, N_{n-1},…,N_0)``.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "wl_oracle.cpp")
_LIB = os.path.join(_HERE, "libwl_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """g++ -O2 -ffp-contract=off (no FMA contraction, IEEE divide)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fno-fast-math",
                               "-shared", "-fPIC", "-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        vp, i32, i64p, f64 = ctypes.c_void_p, ctypes.c_int, ctypes.POINTER(ctypes.c_int64), ctypes.c_double
        f64p, i32p = ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_int)
        L.orc_create.restype, L.orc_create.argtypes = vp, [i32, i64p, i32]
        L.orc_destroy.restype, L.orc_destroy.argtypes = None, [vp]
        L.orc_num_levels.restype, L.orc_num_levels.argtypes = i32, [vp]
        L.orc_level_dims.restype, L.orc_level_dims.argtypes = None, [vp, i32, i64p]
        L.orc_set_coeff.restype, L.orc_set_coeff.argtypes = None, [vp, vp]
        L.orc_get_coeff.restype, L.orc_get_coeff.argtypes = None, [vp, i32, vp]
        L.orc_apply_A.restype, L.orc_apply_A.argtypes = None, [vp, i32, vp, vp]
        L.orc_residual.restype, L.orc_residual.argtypes = f64, [vp, i32, vp, vp, vp]
        L.orc_jacobi.restype, L.orc_jacobi.argtypes = None, [vp, i32, vp, vp, i32]
        L.orc_restrict.restype, L.orc_restrict.argtypes = None, [vp, i32, vp, vp]
        L.orc_prolong_add.restype, L.orc_prolong_add.argtypes = None, [vp, i32, vp, vp]
        L.orc_vcycle_level.restype, L.orc_vcycle_level.argtypes = None, [vp, i32, vp, vp]
        L.orc_vcycle.restype, L.orc_vcycle.argtypes = f64, [vp, vp, vp]
        L.orc_solve.restype, L.orc_solve.argtypes = i32, [vp, vp, vp, f64, i32, f64p, i32p]
        L.orc_project.restype, L.orc_project.argtypes = i32, [vp, vp, vp, vp, f64, i32, f64p, i32p]
        L.orc_mu0.restype, L.orc_mu0.argtypes = f64, [f64]
        L.orc_body_coeff.restype, L.orc_body_coeff.argtypes = i32, [i32, i64p, i32, i32, f64p, vp]
        L.orc_solve_pcg.restype, L.orc_solve_pcg.argtypes = i32, [vp, vp, vp, f64, i32, f64p, i32p]
        L.orc_convdiff.restype, L.orc_convdiff.argtypes = i32, [i32, i64p, i32, vp, f64, vp]
        L.orc_face_value.restype, L.orc_face_value.argtypes = f64, [i32, f64, f64, f64]
        L.orc_divergence.restype, L.orc_divergence.argtypes = None, [vp, vp, vp]
        L.orc_gradient_correct.restype, L.orc_gradient_correct.argtypes = None, [vp, vp, vp]
        L.orc_remove_mean.restype, L.orc_remove_mean.argtypes = None, [vp, vp]
        _lib = L
    return _lib


def _ptr(a: np.ndarray):
    return a.ctypes.data_as(ctypes.c_void_p)


BODY_SPHERE, BODY_TORUS = 0, 1


def body_records(bodies) -> np.ndarray:
    """Pack bodies [(kind, centre, R[, r]), ...] into the 8-doubles-per-body records of orc_body_coeff / wl_set_bodies."""
    rec = np.zeros((len(bodies), 8), dtype=np.float64)
    for k, bd in enumerate(bodies):
        kind, centre, R = bd[0], bd[1], bd[2]
        rec[k, 0] = kind
        rec[k, 1:1 + len(centre)] = centre
        rec[k, 4] = R
        rec[k, 5] = bd[3] if len(bd) > 3 else 0.0
    return rec


def mu0(d: float) -> float:
    return float(lib().orc_mu0(float(d)))


def body_coeff(dims, dtype, bodies) -> np.ndarray:
    """BDIM face coefficients L = mu0(min_k d_k) at the face centres (NEXT-3), walls zeroed; shape (n, N_{n-1}, ..., N_0)."""
    dims = tuple(int(d) for d in dims)
    n = len(dims)
    dt = np.dtype(dtype)
    rec = np.ascontiguousarray(bodies, dtype=np.float64).reshape(-1, 8)
    out = np.empty((n,) + tuple(reversed(dims)), dtype=dt)
    arr = (ctypes.c_int64 * n)(*dims)
    rc = lib().orc_body_coeff(n, arr, 0 if dt == np.float32 else 1, rec.shape[0],
                              rec.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), _ptr(out))
    assert rc == 0
    return out


def face_value(uu: float, c: float, d: float, dtype=np.float64) -> float:
    """Limited third-order face value of (far-upstream, upstream, downstream) (NEXT-4)."""
    return float(lib().orc_face_value(0 if np.dtype(dtype) == np.float32 else 1, float(uu), float(c), float(d)))


def convdiff(u, nu: float) -> np.ndarray:
    """r = convection + diffusion rate of change of the face field u, shape (n, N_{n-1}, ..., N_0) (NEXT-4)."""
    u = np.ascontiguousarray(u)
    assert u.dtype in (np.float32, np.float64)
    n = u.shape[0]
    dims = tuple(reversed(u.shape[1:]))
    assert len(dims) == n
    r = np.empty_like(u)
    arr = (ctypes.c_int64 * n)(*dims)
    rc = lib().orc_convdiff(n, arr, 0 if u.dtype == np.float32 else 1, _ptr(u), float(nu), _ptr(r))
    assert rc == 0
    return r


class Oracle:
    """One grid hierarchy on the host.  ``dims`` is (N_0, …, N_{n-1}), axis 0 unit-stride."""

    def __init__(self, dims, dtype=np.float32):
        self.dims = tuple(int(d) for d in dims)
        self.n = len(self.dims)
        self.dtype = np.dtype(dtype)
        code = {np.dtype(np.float32): 0, np.dtype(np.float64): 1}[self.dtype]
        arr = (ctypes.c_int64 * self.n)(*self.dims)
        self._h = lib().orc_create(self.n, arr, code)
        if not self._h:
            raise ValueError(f"oracle: bad dims {self.dims}")
        self.num_levels = lib().orc_num_levels(self._h)

    def __del__(self):
        if getattr(self, "_h", None):
            lib().orc_destroy(self._h)
            self._h = None

    # -- helpers -------------------------------------------------------------------------------
    def level_dims(self, level: int):
        out = (ctypes.c_int64 * self.n)()
        lib().orc_level_dims(self._h, level, out)
        return tuple(int(v) for v in out)

    def cell_shape(self, level: int = 0):
        return tuple(reversed(self.level_dims(level)))

    def _c(self, a, shape=None):
        a = np.ascontiguousarray(a, dtype=self.dtype)
        if shape is not None:
            assert a.shape == tuple(shape), (a.shape, shape)
        return a

    # -- steps ---------------------------------------------------------------------------------
    def set_coeff(self, L):
        L = self._c(L, (self.n,) + self.cell_shape(0))
        lib().orc_set_coeff(self._h, _ptr(L))

    def get_coeff(self, level: int):
        out = np.empty((self.n,) + self.cell_shape(level), dtype=self.dtype)
        lib().orc_get_coeff(self._h, level, _ptr(out))
        return out

    def apply_A(self, x, level: int = 0):
        x = self._c(x, self.cell_shape(level))
        y = np.empty_like(x)
        lib().orc_apply_A(self._h, level, _ptr(x), _ptr(y))
        return y

    def residual(self, x, b, level: int = 0):
        x = self._c(x, self.cell_shape(level))
        b = self._c(b, self.cell_shape(level))
        r = np.empty_like(x)
        nrm = lib().orc_residual(self._h, level, _ptr(x), _ptr(b), _ptr(r))
        return r, nrm

    def jacobi(self, x, b, sweeps: int, level: int = 0):
        x = self._c(x, self.cell_shape(level)).copy()
        b = self._c(b, self.cell_shape(level))
        lib().orc_jacobi(self._h, level, _ptr(x), _ptr(b), int(sweeps))
        return x

    def restrict(self, r, level: int = 0):
        r = self._c(r, self.cell_shape(level))
        rc = np.empty(self.cell_shape(level + 1), dtype=self.dtype)
        lib().orc_restrict(self._h, level, _ptr(r), _ptr(rc))
        return rc

    def prolong_add(self, xc, xf, level: int = 0):
        xc = self._c(xc, self.cell_shape(level + 1))
        xf = self._c(xf, self.cell_shape(level)).copy()
        lib().orc_prolong_add(self._h, level, _ptr(xc), _ptr(xf))
        return xf

    def vcycle_level(self, x, b, level: int):
        x = self._c(x, self.cell_shape(level)).copy()
        b = self._c(b, self.cell_shape(level))
        lib().orc_vcycle_level(self._h, level, _ptr(x), _ptr(b))
        return x

    def vcycle(self, p, b):
        """One V-cycle + mean removal.  Returns (p_new, ||b - A p_new||inf)."""
        p = self._c(p, self.cell_shape(0)).copy()
        b = self._c(b, self.cell_shape(0))
        nrm = lib().orc_vcycle(self._h, _ptr(p), _ptr(b))
        return p, nrm

    def solve(self, p, b, tol: float, maxcycles: int):
        """Returns (p, hist[0..ncycles], ncycles, rc) with rc = 1 if the cycle cap was reached."""
        p = self._c(p, self.cell_shape(0)).copy()
        b = self._c(b, self.cell_shape(0))
        hist = np.zeros(maxcycles + 1, dtype=np.float64)
        nc = ctypes.c_int(0)
        rc = lib().orc_solve(self._h, _ptr(p), _ptr(b), float(tol), int(maxcycles),
                             hist.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), ctypes.byref(nc))
        return p, hist[: nc.value + 1].copy(), nc.value, rc

    def solve_pcg(self, p, b, tol: float, maxit: int):
        """V-cycle-preconditioned conjugate gradients (NEXT-1).  Returns (p, hist[0..nit], nit, rc)."""
        p = self._c(p, self.cell_shape(0)).copy()
        b = self._c(b, self.cell_shape(0))
        hist = np.zeros(maxit + 1, dtype=np.float64)
        nit = ctypes.c_int(0)
        rc = lib().orc_solve_pcg(self._h, _ptr(p), _ptr(b), float(tol), int(maxit),
                                 hist.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), ctypes.byref(nit))
        return p, hist[: nit.value + 1].copy(), nit.value, rc

    def project(self, u, L, p, tol: float, maxcycles: int):
        """Returns (u_new, p, hist, ncycles, rc).  ``L=None`` keeps the current coefficients."""
        u = self._c(u, (self.n,) + self.cell_shape(0)).copy()
        p = self._c(p, self.cell_shape(0)).copy()
        Lp = None
        if L is not None:
            L = self._c(L, (self.n,) + self.cell_shape(0))
            Lp = _ptr(L)
        hist = np.zeros(maxcycles + 1, dtype=np.float64)
        nc = ctypes.c_int(0)
        rc = lib().orc_project(self._h, _ptr(u), Lp, _ptr(p), float(tol), int(maxcycles),
                               hist.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), ctypes.byref(nc))
        return u, p, hist[: nc.value + 1].copy(), nc.value, rc

    def divergence(self, u):
        u = self._c(u, (self.n,) + self.cell_shape(0))
        b = np.empty(self.cell_shape(0), dtype=self.dtype)
        lib().orc_divergence(self._h, _ptr(u), _ptr(b))
        return b

    def gradient_correct(self, u, p):
        u = self._c(u, (self.n,) + self.cell_shape(0)).copy()
        p = self._c(p, self.cell_shape(0))
        lib().orc_gradient_correct(self._h, _ptr(u), _ptr(p))
        return u

    def remove_mean(self, p):
        p = self._c(p, self.cell_shape(0)).copy()
        lib().orc_remove_mean(self._h, _ptr(p))
        return p
