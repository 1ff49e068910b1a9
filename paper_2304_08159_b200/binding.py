"""Thin Python binding of include/wl.h (ctypes).  Argument marshalling only: every step of the path runs in the
CUDA kernels of libwl.so.  PyTorch is used for device memory and streams — nothing else.

There is NO fallback: if libwl.so is missing or no CUDA device is present, the first call raises.
Functions carry the names of the C entry points and take torch CUDA tensors laid out as include/wl.h says:
cell field ``(N_{n-1},…,N_0)`` contiguous, face field ``(n, N_{n-1},…,N_0)`` contiguous.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libwl.so")

WL_F32, WL_F64 = 0, 1
WL_OK, WL_NOT_CONVERGED = 0, 1
WL_EINVAL, WL_EDIMS, WL_ENOMEM, WL_ECUDA, WL_ESTATE, WL_ENONFINITE = -1, -2, -3, -4, -5, -6
WL_OPT_FUSED, WL_OPT_GRAPH, WL_OPT_COARSE_CTA, WL_OPT_SOLVE_KERNELS, WL_OPT_SOLVER, WL_OPT_HOST_P_ZERO, WL_OPT_PDL = 1, 2, 3, 4, 5, 6, 7

# every symbol include/wl.h declares: (restype, argtypes)
_vp, _i32, _i64, _f64 = ctypes.c_void_p, ctypes.c_int, ctypes.c_int64, ctypes.c_double
_i64p, _f64p, _i32p = ctypes.POINTER(ctypes.c_int64), ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_int)
SIGNATURES = {
    "wl_create": (_i32, [_i32, _i64p, _i32, ctypes.POINTER(_vp)]),
    "wl_destroy": (None, [_vp]),
    "wl_set_stream": (_i32, [_vp, _vp]),
    "wl_set_option": (_i32, [_vp, _i32, _i32]),
    "wl_set_coeff": (_i32, [_vp, _vp]),
    "wl_set_bodies": (_i32, [_vp, _i32, _f64p]),
    "wl_vcycle": (_i32, [_vp, _vp, _vp, _f64p]),
    "wl_solve": (_i32, [_vp, _vp, _vp, _f64, _i32, _f64p, _i32p]),
    "wl_solve_pcg": (_i32, [_vp, _vp, _vp, _f64, _i32, _f64p, _i32p]),
    "wl_project": (_i32, [_vp, _vp, _vp, _vp, _f64, _i32, _f64p, _i32p]),
    "wl_project_host": (_i32, [_vp, _vp, _vp, _vp, _f64, _i32, _f64p, _i32p]),
    "wl_divergence": (_i32, [_vp, _vp, _vp]),
    "wl_gradient": (_i32, [_vp, _vp, _vp]),
    "wl_convdiff": (_i32, [_vp, _vp, _f64, _vp]),
    "wl_jacobi": (_i32, [_vp, _i32, _vp, _vp, _i32]),
    "wl_residual_restrict": (_i32, [_vp, _i32, _vp, _vp, _vp]),
    "wl_prolong_correct": (_i32, [_vp, _i32, _vp, _vp]),
    "wl_down": (_i32, [_vp, _i32, _vp, _vp, _vp, _vp]),
    "wl_up": (_i32, [_vp, _i32, _vp, _vp, _vp, _vp]),
    "wl_vcycle_level": (_i32, [_vp, _i32, _vp, _vp]),
    "wl_residual_norm": (_i32, [_vp, _vp, _vp, _f64p, _f64p]),
    "wl_residual_norm_static": (_i32, [_i32, _i64p, _i32, _vp, _vp, _vp, _vp, _vp]),
    "wl_static_last_error": (ctypes.c_char_p, []),
    "wl_selftest_recip": (_i32, [_vp, ctypes.POINTER(ctypes.c_uint64), ctypes.POINTER(ctypes.c_uint32)]),
    "wl_selftest_fp32_rates": (_i32, [_vp, _f64p]),
    "wl_num_levels": (_i32, [_vp]),
    "wl_level_dims": (_i32, [_vp, _i32, _i64p]),
    "wl_get_coeff": (_i32, [_vp, _i32, _vp]),
    "wl_launch_count": (_i64, [_vp]),
    "wl_plan_fused3d": (_i32, [_i64p, _i32, _i32, _i32, _i32p, _i32, _i32p, _i32p, _i64p]),
    "wl_last_error": (ctypes.c_char_p, [_vp]),
}

_lib = None


class WlError(RuntimeError):
    def __init__(self, code: int, where: str, text: str):
        super().__init__(f"{where} failed with code {code}: {text}")
        self.code = code


def load():
    """Load libwl.so (built in-tree by paper_2304_08159_b200.build).  Raises if it is missing: no fallback."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_2304_08159_b200.build` "
                               "(the CUDA extension is the only implementation; there is no CPU fallback)")
        L = ctypes.CDLL(LIB_PATH)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(L, name)
            fn.restype, fn.argtypes = res, args
        _lib = L
    return _lib


def _check(ctx, rc: int, where: str) -> int:
    if rc < 0:
        raise WlError(rc, where, (load().wl_last_error(ctx) or b"").decode())
    return rc


def _dptr(t, ctx_dtype=None):
    """Device pointer of a contiguous CUDA tensor."""
    if t is None:
        return None
    if not t.is_cuda:
        raise TypeError("expected a CUDA tensor (the library has no CPU path)")
    if not t.is_contiguous():
        raise ValueError("tensor must be contiguous")
    return ctypes.c_void_p(t.data_ptr())


def _dtype_code(dtype) -> int:
    import torch
    if dtype in (torch.float32, np.float32, "float32", "f32", WL_F32):
        return WL_F32
    if dtype in (torch.float64, np.float64, "float64", "f64"):
        return WL_F64
    raise ValueError(f"unsupported dtype {dtype}")


# ---- entry points, same names as include/wl.h ---------------------------------------------------------------------

def wl_create(dims, dtype):
    """dims = (N_0,…,N_{n-1}), axis 0 unit-stride.  Returns an opaque context handle."""
    n = len(dims)
    arr = (ctypes.c_int64 * max(n, 1))(*[int(d) for d in dims])
    out = ctypes.c_void_p()
    rc = load().wl_create(n, arr, _dtype_code(dtype), ctypes.byref(out))
    _check(None, rc, "wl_create")
    return out


def wl_destroy(ctx):
    load().wl_destroy(ctx)


def wl_set_stream(ctx, stream=None):
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return _check(ctx, load().wl_set_stream(ctx, ctypes.c_void_p(s.cuda_stream)), "wl_set_stream")


def wl_set_option(ctx, key: int, value: int):
    return _check(ctx, load().wl_set_option(ctx, int(key), int(value)), "wl_set_option")


def wl_set_coeff(ctx, L):
    return _check(ctx, load().wl_set_coeff(ctx, _dptr(L)), "wl_set_coeff")


WL_BODY_SPHERE, WL_BODY_TORUS = 0, 1


def wl_set_bodies(ctx, records):
    """records: array-like (nbodies, 8) of float64: kind, c0, c1, c2, R, r, 0, 0 (see include/wl.h)."""
    rec = np.ascontiguousarray(records, dtype=np.float64).reshape(-1, 8)
    ptr = rec.ctypes.data_as(_f64p) if rec.shape[0] else None
    return _check(ctx, load().wl_set_bodies(ctx, int(rec.shape[0]), ptr), "wl_set_bodies")


def wl_vcycle(ctx, p, b, want_norm: bool = True):
    out = ctypes.c_double(0.0)
    rc = load().wl_vcycle(ctx, _dptr(p), _dptr(b), ctypes.byref(out) if want_norm else None)
    _check(ctx, rc, "wl_vcycle")
    return out.value if want_norm else None


def wl_solve(ctx, p, b, tol: float, maxcycles: int):
    """Returns (hist[0..ncycles] as float64 ndarray, ncycles, rc)."""
    hist = np.zeros(maxcycles + 1, dtype=np.float64)
    nc = ctypes.c_int(0)
    rc = load().wl_solve(ctx, _dptr(p), _dptr(b), float(tol), int(maxcycles),
                         hist.ctypes.data_as(_f64p), ctypes.byref(nc))
    _check(ctx, rc, "wl_solve")
    return hist[: nc.value + 1].copy(), nc.value, rc


def wl_solve_pcg(ctx, p, b, tol: float, maxit: int):
    """V-cycle-preconditioned conjugate gradients.  Returns (hist[0..nit] as float64 ndarray, nit, rc)."""
    hist = np.zeros(maxit + 1, dtype=np.float64)
    nit = ctypes.c_int(0)
    rc = load().wl_solve_pcg(ctx, _dptr(p), _dptr(b), float(tol), int(maxit), hist.ctypes.data_as(_f64p), ctypes.byref(nit))
    _check(ctx, rc, "wl_solve_pcg")
    return hist[: nit.value + 1].copy(), nit.value, rc


def wl_project(ctx, u, L, p, tol: float, maxcycles: int):
    """In place on u and p.  L=None keeps the current coefficients.  Returns (hist, ncycles, rc)."""
    hist = np.zeros(maxcycles + 1, dtype=np.float64)
    nc = ctypes.c_int(0)
    rc = load().wl_project(ctx, _dptr(u), _dptr(L), _dptr(p), float(tol), int(maxcycles),
                           hist.ctypes.data_as(_f64p), ctypes.byref(nc))
    _check(ctx, rc, "wl_project")
    return hist[: nc.value + 1].copy(), nc.value, rc


def wl_project_host(ctx, u_host, L_host, p_host, tol: float, maxcycles: int):
    """HOST tensors/arrays (pinned torch CPU tensors or NumPy arrays), in place on u_host and p_host."""
    def hptr(a):
        if a is None:
            return None
        if isinstance(a, np.ndarray):
            assert a.flags["C_CONTIGUOUS"]
            return ctypes.c_void_p(a.ctypes.data)
        assert not a.is_cuda and a.is_contiguous()
        return ctypes.c_void_p(a.data_ptr())
    hist = np.zeros(maxcycles + 1, dtype=np.float64)
    nc = ctypes.c_int(0)
    rc = load().wl_project_host(ctx, hptr(u_host), hptr(L_host), hptr(p_host), float(tol), int(maxcycles),
                                hist.ctypes.data_as(_f64p), ctypes.byref(nc))
    _check(ctx, rc, "wl_project_host")
    return hist[: nc.value + 1].copy(), nc.value, rc


def wl_divergence(ctx, u, b):
    return _check(ctx, load().wl_divergence(ctx, _dptr(u), _dptr(b)), "wl_divergence")


def wl_gradient(ctx, u, p):
    return _check(ctx, load().wl_gradient(ctx, _dptr(u), _dptr(p)), "wl_gradient")


def wl_convdiff(ctx, u, nu: float, r):
    return _check(ctx, load().wl_convdiff(ctx, _dptr(u), float(nu), _dptr(r)), "wl_convdiff")


def wl_jacobi(ctx, level: int, x, b, sweeps: int):
    return _check(ctx, load().wl_jacobi(ctx, int(level), _dptr(x), _dptr(b), int(sweeps)), "wl_jacobi")


def wl_residual_restrict(ctx, level: int, x, b, bc):
    return _check(ctx, load().wl_residual_restrict(ctx, int(level), _dptr(x), _dptr(b), _dptr(bc)), "wl_residual_restrict")


def wl_prolong_correct(ctx, level: int, xc, x):
    return _check(ctx, load().wl_prolong_correct(ctx, int(level), _dptr(xc), _dptr(x)), "wl_prolong_correct")


def wl_down(ctx, level: int, x_in, b, x_out, bc=None):
    """x_out = J(J(x_in)) (x_in=None: from zero); bc (None: the context's level+1 rhs) = R(b - A x_out)."""
    return _check(ctx, load().wl_down(ctx, int(level), _dptr(x_in), _dptr(b), _dptr(x_out), _dptr(bc)), "wl_down")


def wl_up(ctx, level: int, x_in, xc, b, x_out):
    """x_out = J(J(x_in + P xc)); xc=None: the context's level+1 iterate."""
    return _check(ctx, load().wl_up(ctx, int(level), _dptr(x_in), _dptr(xc), _dptr(b), _dptr(x_out)), "wl_up")


def wl_vcycle_level(ctx, level: int, x, b):
    return _check(ctx, load().wl_vcycle_level(ctx, int(level), _dptr(x), _dptr(b)), "wl_vcycle_level")


def wl_residual_norm(ctx, p, b):
    """Returns (||b - A p||inf, mean(p))."""
    r, m = ctypes.c_double(0.0), ctypes.c_double(0.0)
    _check(ctx, load().wl_residual_norm(ctx, _dptr(p), _dptr(b), ctypes.byref(r), ctypes.byref(m)), "wl_residual_norm")
    return r.value, m.value


def wl_selftest_recip(ctx):
    """Exhaustive device check of the fused kernels' fp32 reciprocal against IEEE 1/d.  Returns (mismatches, first bad bits)."""
    n, first = ctypes.c_uint64(0), ctypes.c_uint32(0)
    _check(ctx, load().wl_selftest_recip(ctx, ctypes.byref(n), ctypes.byref(first)), "wl_selftest_recip")
    return int(n.value), int(first.value)


def wl_selftest_fp32_rates(ctx) -> dict:
    """Measured fp32 issue and arithmetic rates per clock and SM: {variant: (warp_instr_per_clk, lane_ops_per_clk)}."""
    out = (ctypes.c_double * 8)()
    _check(ctx, load().wl_selftest_fp32_rates(ctx, out), "wl_selftest_fp32_rates")
    names = ("add.f32", "add.f32x2", "fma.f32", "fma.f32x2")
    return {nm: (out[2 * i], out[2 * i + 1]) for i, nm in enumerate(names)}


WL_STATIC_MAX_CELLS = 1 << 27


def wl_residual_norm_static(dims, L, p, b, out, stream=None):
    """Context-free residual check that allocates nothing on the device (include/wl.h): for a caller who has no device
    memory left to request, or no allocator of its own, in the middle of a run.  dims = (N_0,…,N_{n-1}) as in wl_create;
    L, p, b: CUDA tensors of one dtype; out: CUDA float64 tensor of >= 2 elements, receives (||b - A p||inf, mean(p)) when
    the stream has drained.  Enqueued on `stream` (default: torch's current stream).  Grids above WL_STATIC_MAX_CELLS are
    refused.  Calls on one GPU share a fixed scratch array: keep them in stream order."""
    import torch
    if out.dtype != torch.float64 or out.numel() < 2:
        raise ValueError("out must be a float64 CUDA tensor of at least 2 elements")
    if not (L.dtype == p.dtype == b.dtype):
        raise ValueError("L, p, b must share one dtype")
    n = len(dims)
    arr = (ctypes.c_int64 * max(n, 1))(*[int(d) for d in dims])
    s = torch.cuda.current_stream(p.device) if stream is None else stream
    lib = load()
    with torch.cuda.device(p.device):                      # the scratch address is looked up for the CURRENT device
        rc = lib.wl_residual_norm_static(n, arr, _dtype_code(p.dtype), _dptr(L), _dptr(p), _dptr(b), _dptr(out),
                                         ctypes.c_void_p(s.cuda_stream))
    if rc < 0:
        raise WlError(rc, "wl_residual_norm_static", (lib.wl_static_last_error() or b"").decode())
    return rc


def wl_static_last_error() -> str:
    return (load().wl_static_last_error() or b"").decode()


def wl_num_levels(ctx) -> int:
    return _check(ctx, load().wl_num_levels(ctx), "wl_num_levels")


def wl_level_dims(ctx, level: int, ndim: int):
    out = (ctypes.c_int64 * 3)()
    _check(ctx, load().wl_level_dims(ctx, int(level), out), "wl_level_dims")
    return tuple(int(out[i]) for i in range(ndim))


def wl_get_coeff(ctx, level: int, out):
    return _check(ctx, load().wl_get_coeff(ctx, int(level), _dptr(out)), "wl_get_coeff")


def wl_launch_count(ctx) -> int:
    return int(load().wl_launch_count(ctx))


def wl_plan_fused3d(dims, dtype, num_sms: int = 148):
    """Work split of one fused 3-D level half (host only, no GPU): dims = (N_0, N_1, N_2) as in wl_create.
    Returns (items[k] = (X0, Y0, z0, nz), start[grid + 1], load)."""
    d = (ctypes.c_int64 * 3)(*[int(v) for v in dims])
    dt = _dtype_code(dtype)
    grid, load_ = ctypes.c_int(), ctypes.c_int64()
    n = load().wl_plan_fused3d(d, dt, int(num_sms), 0, None, 0, None, ctypes.byref(grid), ctypes.byref(load_))
    if n < 0:
        raise WlError(n, "wl_plan_fused3d", "bad dims / dtype")
    items = (ctypes.c_int * (4 * n))()
    start = (ctypes.c_int * (grid.value + 1))()
    load().wl_plan_fused3d(d, dt, int(num_sms), n, items, grid.value + 1, start, ctypes.byref(grid), ctypes.byref(load_))
    return np.array(items, dtype=np.int64).reshape(n, 4), np.array(start, dtype=np.int64), int(load_.value)


def wl_last_error(ctx) -> str:
    return (load().wl_last_error(ctx) or b"").decode()


class Projector:
    """Convenience owner of one context (create / destroy, stream binding, tensor allocation helpers)."""

    def __init__(self, dims, dtype="float32", device="cuda:0"):
        import torch
        self.dims = tuple(int(d) for d in dims)
        self.n = len(self.dims)
        self.torch_dtype = torch.float32 if _dtype_code(dtype) == WL_F32 else torch.float64
        self.device = torch.device(device)
        if not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: the pressure projection has no CPU path")
        with torch.cuda.device(self.device):
            self.ctx = wl_create(self.dims, self.torch_dtype)
            wl_set_stream(self.ctx)
        self.num_levels = wl_num_levels(self.ctx)

    def close(self):
        if getattr(self, "ctx", None):
            wl_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def cell_shape(self, level: int = 0):
        return tuple(reversed(wl_level_dims(self.ctx, level, self.n)))

    def empty_cells(self, level: int = 0):
        import torch
        return torch.empty(self.cell_shape(level), dtype=self.torch_dtype, device=self.device)

    def zeros_cells(self, level: int = 0):
        import torch
        return torch.zeros(self.cell_shape(level), dtype=self.torch_dtype, device=self.device)

    def empty_faces(self, level: int = 0):
        import torch
        return torch.empty((self.n,) + self.cell_shape(level), dtype=self.torch_dtype, device=self.device)

    def get_coeff(self, level: int):
        out = self.empty_faces(level)
        wl_get_coeff(self.ctx, level, out)
        return out
