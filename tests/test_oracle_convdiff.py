"""Pins of the oracle's convdiff (`convdiff!`; DESIGN.md §3 reading 15).

The paper prints no value of the routine, so the oracle is pinned by what the mathematics fixes: Leonard's normalised-
variable diagram written independently, polynomial exactness of the third-order finite-volume face value, a Kronecker-sum
Laplacian for the diffusive part, convergence to the analytic convection-diffusion term of the Taylor-Green field,
upwinding of a step profile, mirror / axis-permutation covariance and momentum conservation.  None of them retypes the
oracle's loop.
"""
import numpy as np
import pytest

import oracle


# ---- the face value --------------------------------------------------------------------------------------------------------
def nvd(tc: float) -> float:
    """Leonard's universal limiter in normalised variables (far upstream -> 0, downstream -> 1), slope 10, around the
    third-order finite-volume line (2 + 5 tc) / 6.  Outside the monotone range 0 <= tc <= 1: first-order upwind."""
    if tc <= 0.0 or tc >= 1.0:
        return tc
    return max(tc, min((2.0 + 5.0 * tc) / 6.0, 1.0, 10.0 * tc))


def test_face_value_matches_normalised_variable_diagram():
    rng = np.random.default_rng(1)
    for _ in range(4000):
        uu, d = rng.uniform(-3, 3, 2)
        if abs(d - uu) < 1e-3:
            continue
        tc = rng.choice([rng.uniform(-1, 2), rng.uniform(0, 0.12), rng.uniform(0.7, 1.0)])
        c = uu + tc * (d - uu)
        want = uu + nvd(tc) * (d - uu)
        got = oracle.face_value(uu, c, d)
        assert abs(got - want) <= 1e-12 * max(1.0, abs(uu), abs(d)), (uu, c, d, tc)


def test_face_value_is_bounded_by_its_neighbours_and_equals_upwind_at_extrema():
    rng = np.random.default_rng(2)
    for _ in range(4000):
        uu, c, d = rng.uniform(-2, 2, 3)
        f = oracle.face_value(uu, c, d)
        assert min(c, d) - 1e-15 <= f <= max(c, d) + 1e-15
        if (c - uu) * (d - c) <= 0:   # c is a local extremum: first-order upwind
            assert f == c


def test_face_value_is_exact_for_quadratics_given_by_cell_averages():
    """Three unit cells [-2,-1], [-1,0], [0,1] with averages of q(x) = a + b x + c x^2; the face at x = 0 carries q(0) = a.
    Averages: q over [s, s+1] = a + b (s + 1/2) + c (s^2 + s + 1/3).  Mild curvature keeps the limiter inactive."""
    rng = np.random.default_rng(3)
    for _ in range(200):
        a, b = rng.uniform(-1, 1), rng.uniform(0.5, 1.5) * rng.choice([-1, 1])
        c = rng.uniform(-0.1, 0.1)
        avg = lambda s: a + b * (s + 0.5) + c * (s * s + s + 1.0 / 3.0)
        f = oracle.face_value(avg(-2), avg(-1), avg(0))
        assert abs(f - a) < 1e-14


def test_fp32_face_value_rounds_the_same_formula():
    rng = np.random.default_rng(4)
    for _ in range(500):
        uu, c, d = rng.uniform(-2, 2, 3).astype(np.float32)
        f32 = oracle.face_value(uu, c, d, np.float32)
        f64 = oracle.face_value(float(uu), float(c), float(d))
        assert abs(f32 - f64) <= 4e-6 * max(1.0, abs(float(uu)), abs(float(c)))


# ---- diffusion: r(nu = 1) - r(nu = 0) is the Laplacian with free-slip, impermeable walls -----------------------------------
def lap_component(ui: np.ndarray, axis_normal: int) -> np.ndarray:
    """Second differences of one face component (array axes reversed: array axis a <-> grid axis n-1-a).  Normal axis: the
    stored plane 0 and the unstored plane N are walls (value 0, no equation on plane 0); tangential axes: zero normal
    derivative (mirror)."""
    n = ui.ndim
    out = np.zeros_like(ui)
    for ax in range(n):
        grid_axis = n - 1 - ax
        if grid_axis == axis_normal:
            pad = [(0, 0)] * n
            pad[ax] = (1, 1)
            w = np.pad(ui, pad, mode="constant")          # value 0 beyond both ends (index -1 is never used: plane 0 is masked)
        else:
            pad = [(0, 0)] * n
            pad[ax] = (1, 1)
            w = np.pad(ui, pad, mode="edge")               # mirror: zero flux through the wall
        sl = lambda a, b: tuple(slice(a, b) if k == ax else slice(None) for k in range(n))
        m = ui.shape[ax]
        out += w[sl(2, m + 2)] - 2.0 * w[sl(1, m + 1)] + w[sl(0, m)]
    idx = [slice(None)] * n
    idx[n - 1 - axis_normal] = 0
    out[tuple(idx)] = 0.0
    return out


@pytest.mark.parametrize("shape", [(10, 12), (6, 8, 10)])
def test_diffusive_part_is_the_free_slip_laplacian(shape):
    n = len(shape)
    rng = np.random.default_rng(5)
    u = rng.standard_normal((n,) + shape)
    for i in range(n):                       # wall planes hold the wall value
        idx = [slice(None)] * n
        idx[n - 1 - i] = 0
        u[(i,) + tuple(idx)] = 0.0
    d = oracle.convdiff(u, 1.0) - oracle.convdiff(u, 0.0)
    for i in range(n):
        want = lap_component(u[i], i)
        assert np.max(np.abs(d[i] - want)) < 1e-12, i


# ---- the whole operator converges to -(u.grad)u + nu lap u on the Taylor-Green field (closed free-slip box) -------------------
def tgv(N: int, n: int):
    """Face-centred samples of u = (sin x cos y cos z, -cos x sin y cos z, 0) on [0, 2 pi]^n (n = 2: z dropped) and the
    analytic r = -(u.grad)u + nu lap u at the same points."""
    h = 2 * np.pi / N
    c = (np.arange(N) + 0.5) * h
    f = np.arange(N) * h
    u = np.zeros((n,) + (N,) * n)
    r = np.zeros_like(u)
    nu = 0.05
    k2 = float(n)                    # lap u = -n u for these modes
    for i in range(2):
        axes = [f if a == i else c for a in range(n)]           # grid axes 0..n-1
        X = np.meshgrid(*axes[::-1], indexing="ij")[::-1]       # X[a] varies along array axis n-1-a
        x, y = X[0], X[1]
        cz = np.cos(X[2]) if n == 3 else 1.0
        if i == 0:
            u[0] = np.sin(x) * np.cos(y) * cz
            conv = np.sin(x) * np.cos(x) * cz * cz               # u u_x + v u_y (+ w u_z = 0)
        else:
            u[1] = -np.cos(x) * np.sin(y) * cz
            conv = np.sin(y) * np.cos(y) * cz * cz
        r[i] = -conv - nu * k2 * u[i]
    if n == 3:   # third component: w = 0, but (u.grad) w = 0 and lap w = 0 as well
        pass
    return u, r, nu


@pytest.mark.parametrize("n", [2, 3])
def test_second_order_convergence_on_taylor_green(n):
    errs = []
    for N in (16, 32):
        u, want, nu = tgv(N, n)
        h = 2 * np.pi / N
        # grid units: velocities in cells per unit time -> scale u by 1/h, nu by 1/h^2, r by 1/h
        got = oracle.convdiff(u / h, nu / (h * h)) * h
        e = got - want
        for i in range(n):                    # no equation on the stored wall plane
            idx = [slice(None)] * n
            idx[n - 1 - i] = 0
            e[i][tuple(idx)] = 0.0
        errs.append((np.mean(np.abs(e)), np.max(np.abs(e))))
    # Second order in the mean: the error drops ~4x per halving (measured 3.5).  The limiter falls back to first-order
    # upwind at the O(1) extrema of the field, so the MAXIMUM error is only first order there (measured 2.6x per halving).
    assert errs[0][0] < 0.02 and errs[1][0] < errs[0][0] / 3.2, errs
    assert errs[1][1] < errs[0][1] / 2.0 and errs[0][1] < 0.05, errs


# ---- upwinding -----------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("sign", [1.0, -1.0])
def test_step_profile_moves_downstream_only(sign):
    """2-D, uniform advecting velocity U along axis 0 (interior), u_1 a step in x_0.  The limited scheme reduces to first-order
    upwind at the foot of a step, so exactly one column changes: the first one behind the front as seen by the flow."""
    N0, N1 = 24, 8
    U = 0.75 * sign
    u = np.zeros((2, N1, N0))
    u[0, :, 1:] = U                      # plane 0 is the wall; the profile is read far from the walls only
    u[1, 1:, :12] = 0.0
    u[1, 1:, 12:] = 1.0
    r = oracle.convdiff(u, 0.0)
    col = r[1, 4, 6:18]
    want = np.zeros(12)
    if sign > 0:
        want[12 - 6] = -abs(U)           # the first "1" column loses what flows out of it; nothing flows in from the "0" side
    else:
        want[11 - 6] = +abs(U)           # flow towards -x: the last "0" column fills up
    assert np.allclose(col, want, atol=1e-14), col


# ---- symmetries ----------------------------------------------------------------------------------------------------------------
def random_box_field(shape, rng, zero_near_walls=False):
    n = len(shape)
    u = rng.standard_normal((n,) + shape)
    for i in range(n):
        idx = [slice(None)] * n
        idx[n - 1 - i] = 0
        u[(i,) + tuple(idx)] = 0.0
        if zero_near_walls:
            idx[n - 1 - i] = 1
            u[(i,) + tuple(idx)] = 0.0
            idx[n - 1 - i] = -1
            u[(i,) + tuple(idx)] = 0.0
    return u


def test_axis_permutation_covariance():
    """Swapping grid axes 0 and 1 (and the components with them) swaps the result the same way."""
    rng = np.random.default_rng(7)
    u = random_box_field((6, 7, 9), rng)                      # array (3, N2, N1, N0)
    r = oracle.convdiff(u, 0.3)
    us = np.ascontiguousarray(np.stack([u[1], u[0], u[2]]).transpose(0, 1, 3, 2))
    rs = oracle.convdiff(us, 0.3)
    back = np.stack([rs[1], rs[0], rs[2]]).transpose(0, 1, 3, 2)
    assert np.max(np.abs(back - r)) < 1e-12
    # and axes 0 and 2
    us = np.ascontiguousarray(np.stack([u[2], u[1], u[0]]).transpose(0, 3, 2, 1))
    rs = oracle.convdiff(us, 0.3)
    back = np.stack([rs[2], rs[1], rs[0]]).transpose(0, 3, 2, 1)
    assert np.max(np.abs(back - r)) < 1e-12


def test_mirror_covariance():
    """Reflecting the box along axis 0: face k of the normal component maps to face N - k with the opposite sign (the stored
    wall plane maps to the unstored one), tangential components are flipped cell-wise."""
    rng = np.random.default_rng(8)
    u = random_box_field((6, 8, 10), rng)
    N0 = u.shape[-1]

    def mirror(w):
        m = np.empty_like(w)
        m[0, ..., 0] = 0.0
        m[0, ..., 1:] = -w[0, ..., :0:-1]      # face k <- -face N0-k, k = 1..N0-1
        m[1] = w[1, ..., ::-1]
        m[2] = w[2, ..., ::-1]
        return m

    r = oracle.convdiff(u, 0.2)
    rm = oracle.convdiff(mirror(u), 0.2)
    assert np.max(np.abs(rm - mirror(r))) < 1e-12
    assert N0 == 10


@pytest.mark.parametrize("shape", [(9, 11), (6, 7, 8)])
def test_momentum_is_conserved_when_nothing_touches_the_walls(shape):
    """All fluxes through the walls vanish (tangential: by definition; normal: when the normal velocity is zero on the two
    face planes next to each wall), so the interior flux differences telescope to zero for every component."""
    rng = np.random.default_rng(9)
    u = random_box_field(shape, rng, zero_near_walls=True)
    r = oracle.convdiff(u, 0.1)
    scale = np.sum(np.abs(r))
    for i in range(len(shape)):
        assert abs(np.sum(r[i])) < 1e-13 * scale


def test_wall_planes_are_zero_and_fp32_follows_fp64():
    rng = np.random.default_rng(10)
    u = random_box_field((5, 6, 7), rng)
    r64 = oracle.convdiff(u, 0.1)
    r32 = oracle.convdiff(u.astype(np.float32), 0.1)
    assert r32.dtype == np.float32
    assert np.all(r64[0][..., 0] == 0) and np.all(r64[1][:, 0, :] == 0) and np.all(r64[2][0] == 0)
    assert np.max(np.abs(r32 - r64)) < 2e-4 * np.max(np.abs(r64))
