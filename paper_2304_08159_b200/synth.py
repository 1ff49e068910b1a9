"""Seeded synthetic inputs (L, u) for the pressure-projection path.

This module serves BOTH the CPU oracle (``oracle/``) and the CUDA library, because what it
produces are INPUTS: the face-coefficient field ``L`` and the face-velocity field ``u``.  It holds
none of the method's arithmetic (no operator, no smoother, no transfer, no divergence) and imports
neither the oracle nor the CUDA binding.  NumPy only.

Recipe (BASELINE.json ``configs``):

* Layout: a cell field has NumPy shape ``(N_{n-1}, …, N_0)`` (axis 0 of the problem is the LAST,
  unit-stride, NumPy axis); a face field has shape ``(n, N_{n-1}, …, N_0)``, component slowest.
  Face ``(I, i)`` is the LOWER face of cell ``I`` in direction ``i`` (the printed
  ``u[I,i] -= coeff[I,i]*(p[I]-p[I-del(i)])`` kernel), so plane ``I_i = 0`` is a domain wall.
* Coordinates (cell units): cell ``I`` spans ``[I_i, I_i+1]``; face ``(I, i)`` has coordinate
  ``I_i`` along ``i`` and ``I_j + 1/2`` along every other axis ``j``.
* BDIM coefficient (BASELINE.json north_star): ``L = mu0(d)``, ``d`` = signed distance to the body
  in cells at the face centre, positive in the fluid; evaluated in fp64, clamped to [0, 1], cast.
* Random numbers: counter-based (stateless) splitmix64 hash of ``(seed, linear index)``;
  ``U(-1,1) = (2k+1)/2^24 - 1`` from the top 24 hash bits (exact in fp32, never 0 or +-1);
  ``N(0, sigma)`` by Box-Muller in fp64 from two further hashes of the same counter.
* Seeds: ``230408159 + 1000*config + stream`` (stream 0 = u, 1 = noise, 2 = sphere parameters).
"""
from __future__ import annotations

import math

import numpy as np

SEED0 = 230408159

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)
_GOLD = np.uint64(0x9E3779B97F4A7C15)
_C1 = np.uint64(0xBF58476D1CE4E5B9)
_C2 = np.uint64(0x94D049BB133111EB)


def seed_for(config: int, stream: int) -> int:
    return SEED0 + 1000 * int(config) + int(stream)


def _mix64(z: np.ndarray) -> np.ndarray:
    """splitmix64 finaliser on a uint64 array (wrap-around arithmetic)."""
    with np.errstate(over="ignore"):
        z = (z ^ (z >> np.uint64(30))) * _C1
        z = (z ^ (z >> np.uint64(27))) * _C2
        z = z ^ (z >> np.uint64(31))
    return z


def hash_u64(seed: int, start: int, count: int, lane: int = 0) -> np.ndarray:
    """64 hash bits for counters ``start .. start+count-1`` of stream ``(seed, lane)``."""
    idx = np.arange(start, start + count, dtype=np.uint64)
    with np.errstate(over="ignore"):
        key = _mix64(np.uint64(seed & 0xFFFFFFFFFFFFFFFF) * _GOLD + np.uint64(lane) * _C2 + np.uint64(1))
        z = (idx + np.uint64(1)) * _GOLD + key
    return _mix64(z)


def uniform_pm1(seed: int, count: int, start: int = 0, dtype=np.float32, chunk: int = 1 << 24) -> np.ndarray:
    """``U(-1,1)`` on the 2^24-point odd lattice ``(2k+1)/2^24 - 1`` (exact in fp32)."""
    out = np.empty(count, dtype=dtype)
    for s in range(0, count, chunk):
        c = min(chunk, count - s)
        k = (hash_u64(seed, start + s, c) >> np.uint64(40)).astype(np.int64)
        out[s:s + c] = ((2 * k + 1).astype(np.float64) / float(1 << 24) - 1.0).astype(dtype)
    return out


def normal(seed: int, count: int, sigma: float, start: int = 0, chunk: int = 1 << 23) -> np.ndarray:
    """``N(0, sigma)`` in fp64 by Box-Muller; two independent hash lanes per counter."""
    out = np.empty(count, dtype=np.float64)
    for s in range(0, count, chunk):
        c = min(chunk, count - s)
        a = (hash_u64(seed, start + s, c, lane=1) >> np.uint64(11)).astype(np.float64)
        b = (hash_u64(seed, start + s, c, lane=2) >> np.uint64(11)).astype(np.float64)
        u1 = (a + 0.5) / float(1 << 53)
        u2 = (b + 0.5) / float(1 << 53)
        out[s:s + c] = sigma * np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * math.pi * u2)
    return out


# ------------------------------------------------------------------------------------------------
# BDIM coefficient
# ------------------------------------------------------------------------------------------------

def mu0(d) -> np.ndarray:
    """Zeroth kernel moment of BDIM with eps = 1 (BASELINE.json north_star "BDIM face coefficient").

    0 for d <= -1, 1 for d >= 1, else 0.5*(1 + d + sin(pi d)/pi); evaluated in fp64 and clamped to
    [0, 1] AFTER the formula (the formula is not applied to a clamped d: sin(-pi) != 0 in floating
    point would give a slightly negative coefficient).
    """
    d = np.asarray(d, dtype=np.float64)
    v = 0.5 * (1.0 + d + np.sin(math.pi * d) / math.pi)
    v = np.clip(v, 0.0, 1.0)
    v = np.where(d <= -1.0, 0.0, v)
    v = np.where(d >= 1.0, 1.0, v)
    return v


def _np_shape(dims) -> tuple:
    return tuple(int(x) for x in reversed(dims))


def face_axes(dims, i, lo=None, hi=None):
    """Open-mesh fp64 coordinate vectors (one per problem axis, broadcastable in NumPy axis order)
    of the centres of faces ``(I, i)`` for ``lo <= I < hi``."""
    n = len(dims)
    lo = [0] * n if lo is None else lo
    hi = list(dims) if hi is None else hi
    axes = []
    for j in range(n):
        c = np.arange(lo[j], hi[j], dtype=np.float64)
        if j != i:
            c = c + 0.5
        shape = [1] * n
        shape[n - 1 - j] = c.size
        axes.append(c.reshape(shape))
    return axes


def zero_walls(L: np.ndarray) -> np.ndarray:
    """Set the stored domain-wall plane ``I_i = 0`` of every component to 0 (Neumann walls)."""
    n = L.shape[0]
    for i in range(n):
        idx = [slice(None)] * n
        idx[n - 1 - i] = 0
        L[(i,) + tuple(idx)] = 0
    return L


def coeff_uniform(dims, dtype=np.float32) -> np.ndarray:
    n = len(dims)
    L = np.ones((n,) + _np_shape(dims), dtype=dtype)
    return zero_walls(L)


def coeff_spheres(dims, centres, radii, dtype=np.float32, brute_force: bool = False) -> np.ndarray:
    """``L = mu0(min_k |x - c_k| - R_k)`` at face centres, walls zeroed.

    ``mu0(d) = 1`` exactly for ``d >= 1``, so only faces inside the bounding box (radius + 2 cells)
    of some sphere are evaluated; ``brute_force=True`` evaluates every face (test of equivalence).
    In 2-D a "sphere" is a circle (the cylinder of config 1).
    """
    n = len(dims)
    centres = np.asarray(centres, dtype=np.float64).reshape(-1, n)
    radii = np.asarray(radii, dtype=np.float64).reshape(-1)
    L = np.ones((n,) + _np_shape(dims), dtype=dtype)
    for i in range(n):
        if brute_force:
            ax = face_axes(dims, i)
            d = np.full(_np_shape(dims), np.inf)
            for c, R in zip(centres, radii):
                r2 = sum((ax[j] - c[j]) ** 2 for j in range(n))
                d = np.minimum(d, np.sqrt(r2) - R)
            L[i] = mu0(d).astype(dtype)
            continue
        boxes = []
        for c, R in zip(centres, radii):
            lo = [max(0, int(math.floor(c[j] - R - 2.0))) for j in range(n)]
            hi = [min(int(dims[j]), int(math.ceil(c[j] + R + 2.0)) + 1) for j in range(n)]
            if any(h <= l for l, h in zip(lo, hi)):
                continue
            boxes.append((lo, hi))
        # distance to ALL spheres inside every box (another sphere may be nearer there)
        for lo, hi in boxes:
            ax = face_axes(dims, i, lo, hi)
            d = None
            for c, R in zip(centres, radii):
                # skip spheres that cannot be within distance 1 of this box
                far = False
                for j in range(n):
                    gap = max(lo[j] - 0.5 - c[j], c[j] - (hi[j] + 0.5), 0.0)
                    if gap > R + 1.5:
                        far = True
                        break
                if far:
                    continue
                r2 = sum((ax[j] - c[j]) ** 2 for j in range(n))
                dk = np.sqrt(r2) - R
                d = dk if d is None else np.minimum(d, dk)
            sl = tuple(slice(lo[j], hi[j]) for j in reversed(range(n)))
            L[i][sl] = mu0(d).astype(dtype)
    return zero_walls(L)


def coeff_torus(dims, centre, R: float, r: float, dtype=np.float32) -> np.ndarray:
    """``L = mu0(d)`` for a torus whose axis is the flow axis 0: major radius ``R`` (in the 1-2 plane), minor radius
    ``r``, ``d = sqrt((sqrt(y^2 + z^2) - R)^2 + x^2) - r`` about ``centre``; face centres, fp64, walls zeroed."""
    assert len(dims) == 3
    L = np.empty((3,) + _np_shape(dims), dtype=dtype)
    for i in range(3):
        ax = face_axes(dims, i)
        x, y, z = (ax[j] - float(centre[j]) for j in range(3))
        rho = np.sqrt(y * y + z * z) - float(R)
        d = np.sqrt(rho * rho + x * x) - float(r)
        L[i] = mu0(d).astype(dtype)
    return zero_walls(L)


# ------------------------------------------------------------------------------------------------
# velocity fields
# ------------------------------------------------------------------------------------------------

def velocity_uniform(dims, seed: int, dtype=np.float32) -> np.ndarray:
    """Seeded i.i.d. ``U(-1,1)`` per face, counter = linear face index (component slowest)."""
    n = len(dims)
    M = int(np.prod(dims))
    return uniform_pm1(seed, n * M, dtype=dtype).reshape((n,) + _np_shape(dims))


def velocity_taylor_green(dims, noise_seed: int, sigma: float = 1e-2, dtype=np.float32) -> np.ndarray:
    """Taylor-Green ``u = (sin x cos y cos z, -cos x sin y cos z, 0)`` on ``[0, 2 pi)^3`` sampled at
    face centres (``x_i = 2 pi / N_i *`` cell-unit coordinate) plus seeded ``N(0, sigma)`` noise on
    every face velocity (the noise goes on the FACE VELOCITIES, so that
    the divergence stays mean-zero by construction)."""
    n = len(dims)
    assert n == 3
    M = int(np.prod(dims))
    u = np.empty((n,) + _np_shape(dims), dtype=dtype)
    for i in range(n):
        ax = face_axes(dims, i)
        x, y, z = (ax[j] * (2.0 * math.pi / dims[j]) for j in range(3))
        if i == 0:
            f = np.sin(x) * np.cos(y) * np.cos(z)
        elif i == 1:
            f = -np.cos(x) * np.sin(y) * np.cos(z)
        else:
            f = np.zeros(_np_shape(dims))
        f = f + normal(noise_seed, M, sigma, start=i * M).reshape(_np_shape(dims))
        u[i] = f.astype(dtype)
    return u


# ------------------------------------------------------------------------------------------------
# BASELINE.json configs
# ------------------------------------------------------------------------------------------------

CONFIG_NAMES = {
    0: "cfg0_2d_64x64_uniform",
    1: "cfg1_2d_1024x1024_cylinder",
    2: "cfg2_3d_128^3_sphere",
    3: "cfg3_3d_256^3_uniform_taylor_green",
    4: "cfg4_3d_512^3_32_spheres",
}


def sphere_params(config: int, dims, count: int = 32, rmin: float = 8.0, rmax: float = 32.0,
                  margin: float = 32.0, scale: int = 1):
    """32 seeded spheres: radius U(8,32) cells, centres uniform inside a 32-cell margin (config 4).
    ``scale`` shrinks radii and margin with the grid for reduced-size test cases."""
    n = len(dims)
    seed = seed_for(config, 2)
    r01 = (uniform_pm1(seed, count * (n + 1), dtype=np.float64) + 1.0) * 0.5
    r01 = r01.reshape(count, n + 1)
    radii = (rmin + (rmax - rmin) * r01[:, 0]) / scale
    m = margin / scale
    centres = np.stack([m + (dims[j] - 2 * m) * r01[:, 1 + j] for j in range(n)], axis=1)
    return centres, radii


def body_records(kind: int, centres, radii, tube_radii=None) -> np.ndarray:
    """The analytic bodies of a config as the 8-doubles-per-body records of ``wl_set_bodies`` (include/wl.h): kind (0 sphere
    / circle, 1 torus about axis 0), c0, c1, c2, R, r, 0, 0.  A description of the INPUT geometry, no arithmetic."""
    centres = np.asarray(centres, dtype=np.float64)
    centres = centres.reshape(-1, centres.shape[-1])
    rec = np.zeros((centres.shape[0], 8), dtype=np.float64)
    rec[:, 0] = kind
    rec[:, 1:1 + centres.shape[1]] = centres
    rec[:, 4] = np.asarray(radii, dtype=np.float64).reshape(-1)
    if tube_radii is not None:
        rec[:, 5] = np.asarray(tube_radii, dtype=np.float64).reshape(-1)
    return rec


def make_config(config: int, dtype=None, scale: int = 1) -> dict:
    """Inputs of BASELINE.json ``configs[config]``; ``scale`` (a power of two) divides every grid
    extent and every body length by the same factor for reduced-size parity cases.

    Returns ``dims`` (axis 0 first), ``L`` (walls zeroed), ``u`` (= L * u_raw: the BDIM-masked
    velocity handed to ``wl_project``), ``tol``, ``maxcycles``, ``call``.
    The right-hand side ``b`` is NOT produced here: it is the divergence of ``u``, a step of the
    method (H1), computed by the oracle and by the CUDA library each on their own.
    """
    dt = np.dtype(np.float32 if dtype is None else dtype)
    s = int(scale)
    if config == 0:
        dims = (64 // s, 64 // s)
        L = coeff_uniform(dims, dt)
        bodies = np.zeros((0, 8))
        u = velocity_uniform(dims, seed_for(0, 0), dt)
        tol, maxc, call = 0.0, 10, "solve"
    elif config == 1:
        dims = (1024 // s, 1024 // s)
        L = coeff_spheres(dims, [[256.0 / s, 512.0 / s]], [64.0 / s], dt)
        bodies = body_records(0, [[256.0 / s, 512.0 / s]], [64.0 / s])
        u = velocity_uniform(dims, seed_for(1, 0), dt)
        tol, maxc, call = 1e-4, 32, "solve"
    elif config == 2:
        dims = (128 // s,) * 3
        L = coeff_spheres(dims, [[48.0 / s, 64.0 / s, 64.0 / s]], [24.0 / s], dt)
        bodies = body_records(0, [[48.0 / s, 64.0 / s, 64.0 / s]], [24.0 / s])
        u = velocity_uniform(dims, seed_for(2, 0), dt)
        tol, maxc, call = 1e-4, 32, "project"
    elif config == 3:
        dims = (256 // s,) * 3
        L = coeff_uniform(dims, dt)
        bodies = np.zeros((0, 8))
        u = velocity_taylor_green(dims, seed_for(3, 1), 1e-2, dt)
        tol, maxc, call = 1e-4, 32, "solve"
    elif config == 4:
        dims = (512 // s,) * 3
        centres, radii = sphere_params(4, dims, scale=s)
        L = coeff_spheres(dims, centres, radii, dt)
        bodies = body_records(0, centres, radii)
        u = velocity_uniform(dims, seed_for(4, 0), dt)
        tol, maxc, call = 1e-4, 32, "project"
    else:
        raise ValueError(f"unknown config {config}")
    u *= L  # BDIM-masked velocity (stationary body); walls get u = 0
    return dict(config=config, name=CONFIG_NAMES[config] + (f"_div{s}" if s != 1 else ""),
                dims=dims, dtype=dt, L=L, u=u, tol=tol, maxcycles=maxc, call=call, bodies=bodies)


def make_donut(p: int, dtype=None) -> dict:
    """The paper's second workload shape ("flow past a donut ... N = (2^(p+1), 2^p, 2^p)", p = 4..7):
    a torus in a 2:1:1 box.  The paper gives neither radii nor position; chosen here (and stated in DESIGN.md §5):
    centre (2^p, 2^(p-1), 2^(p-1)) = the box centre, major radius 2^p / 4, minor radius 2^p / 16 cells, axis along
    the long (flow) axis.  Velocity as in config 0 (seeded U(-1,1) per face, masked by L); wl_project to 1e-4."""
    dt = np.dtype(np.float32 if dtype is None else dtype)
    n1 = 1 << int(p)
    dims = (2 * n1, n1, n1)
    L = coeff_torus(dims, (n1, n1 / 2, n1 / 2), n1 / 4.0, n1 / 16.0, dt)
    u = velocity_uniform(dims, seed_for(5, int(p)), dt)
    u *= L
    return dict(config=5, name=f"donut_p{int(p)}_{dims[0]}x{dims[1]}x{dims[2]}", dims=dims, dtype=dt, L=L, u=u,
                tol=1e-4, maxcycles=32, call="project", bodies=body_records(1, [[n1, n1 / 2, n1 / 2]], [n1 / 4.0], [n1 / 16.0]))
