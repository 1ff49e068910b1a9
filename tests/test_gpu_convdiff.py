"""NEXT-4 — wl_convdiff (the paper's `convdiff!`; DESIGN.md §3 reading 15) against the oracle's convdiff,
face by face, through the C ABI.

Bar: every operation of the routine rounds separately on both sides and in the same order (no contraction, IEEE division by
6 — the fp32 kernel's multiply-and-correct quotient is the IEEE one, tests/test_div6.py), the limiter's medians pick a value
out of their arguments, so for finite fields the results are EQUAL as numbers (`np.array_equal`; only the sign of an exact zero
may differ) in fp32 and in fp64.  Shapes: sub-tile, several tiles with ragged tails in x / y and several z-chunks (tiled
kernel: 3-D, rows of whole 16-byte vectors), odd extents and 2-D (one-thread-per-cell kernel), both kernels on the same
input (WL_OPT_FUSED 0 / 1), the full 256^3 and 512^3 fields of configs 3 and 4.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

SHAPES = [(8, 8, 8), (12, 10, 6), (128, 8, 8), (136, 24, 20), (256, 40, 12), (64, 64, 64), (132, 17, 9), (16, 4, 4), (128, 64, 64),
          (13, 9, 7), (6, 5, 4), (64, 64), (33, 17), (256, 24)]
DTYPES = [np.float32, np.float64]


@pytest.fixture(scope="module")
def env(oracle_mod):
    import torch
    from paper_2304_08159_b200 import binding as wl, build
    build.build_cuda()
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return dict(torch=torch, wl=wl, oracle=oracle_mod)


def _field(dims, dt, seed, kind):
    n = len(dims)
    shape = (n,) + tuple(reversed(dims))
    rng = np.random.default_rng(seed)
    if kind == "noise":            # rough: the limiter is active on most faces, U changes sign from face to face
        u = rng.uniform(-1.0, 1.0, shape)
    elif kind == "smooth":         # smooth + small noise: mostly the unlimited third-order branch
        ax = [np.arange(d) for d in reversed(dims)]
        g = np.meshgrid(*ax, indexing="ij")
        u = np.stack([np.sin(0.3 * g[(i + 1) % n] + i) * np.cos(0.2 * g[i] - 0.5 * i) for i in range(n)])
        u = u + 1e-3 * rng.standard_normal(shape)
    else:                          # plateaus: exact ties and exact zeros in the medians, one-signed advection
        u = np.round(rng.uniform(-1.0, 1.0, shape) * 2.0) / 2.0 + 0.25
    return np.ascontiguousarray(u.astype(dt))


def _gpu(env, dims, dt, u, nu, fused):
    torch, wl = env["torch"], env["wl"]
    pr = wl.Projector(dims, dt)
    wl.wl_set_option(pr.ctx, wl.WL_OPT_FUSED, fused)
    ud = torch.from_numpy(u).cuda()
    keep = ud.clone()
    rd = torch.full_like(ud, float("nan"))
    n0 = wl.wl_launch_count(pr.ctx)
    wl.wl_convdiff(pr.ctx, ud, nu, rd)
    torch.cuda.synchronize()
    assert wl.wl_launch_count(pr.ctx) == n0 + 1          # one kernel
    assert torch.equal(ud, keep)                         # u is read-only
    out = rd.cpu().numpy()
    pr.close()
    return out


@pytest.mark.parametrize("dims", SHAPES, ids=lambda d: "x".join(map(str, d)))
@pytest.mark.parametrize("dt", DTYPES, ids=["f32", "f64"])
@pytest.mark.parametrize("kind", ["noise", "smooth", "plateau"])
def test_convdiff_equals_oracle(env, dims, dt, kind):
    u = _field(dims, dt, 7 + dims[0] + 31 * len(dims), kind)   # wall planes left non-zero on purpose: they are read as stored
    for nu in (0.0, 0.0375):
        ref = env["oracle"].convdiff(u, nu)
        for fused in (0, 1):
            got = _gpu(env, dims, dt, u, nu, fused)
            assert np.isfinite(got).all()
            assert np.array_equal(got, ref), (dims, dt, kind, nu, fused, float(np.abs(got - ref).max()))
            for i in range(len(dims)):                         # the stored wall plane of every component is exactly zero
                sl = [slice(None)] * len(dims)
                sl[len(dims) - 1 - i] = 0
                assert not got[i][tuple(sl)].any()


def test_convdiff_tiny_and_huge_magnitudes(env):
    """The multiply-and-correct quotient falls back to the division below 2^-100; scaling the field by powers of two must scale
    the convective part by the square exactly (nu = 0), through the subnormal range as well."""
    dims = (136, 24, 20)
    u = _field(dims, np.float32, 5, "noise")
    for scale in (2.0 ** -40, 2.0 ** -55, 2.0 ** -70, 2.0 ** 30):
        us = (u * np.float32(scale)).astype(np.float32)
        ref = env["oracle"].convdiff(us, 0.0)
        got = _gpu(env, dims, np.float32, us, 0.0, 1)
        assert np.array_equal(got, ref), scale


def test_convdiff_taylor_green_256_full(env):
    """Config 3's velocity (Taylor-Green + N(0, 1e-2) noise) at FULL size, fp32 and fp64, the launch configuration bench.py
    times: every face against the oracle."""
    from paper_2304_08159_b200 import synth
    for dt in DTYPES:
        cfg = synth.make_config(3, dtype=dt)
        u = np.ascontiguousarray(cfg["u"])
        ref = env["oracle"].convdiff(u, 1e-3)
        got = _gpu(env, cfg["dims"], dt, u, 1e-3, 1)
        assert np.array_equal(got, ref)


def test_convdiff_config4_512_full(env):
    """Config 4's masked velocity (512^3 fp32, 32 spheres: zero inside the bodies, so exact zeros and ties abound) at FULL size:
    every face against the oracle (the oracle needs ~2 minutes)."""
    from paper_2304_08159_b200 import synth
    cfg = synth.make_config(4)
    u = np.ascontiguousarray(cfg["u"])
    ref = env["oracle"].convdiff(u, 1e-3)
    got = _gpu(env, cfg["dims"], np.float32, u, 1e-3, 1)
    assert np.array_equal(got, ref)


def test_convdiff_is_reproducible_run_to_run(env):
    """The tiled kernel hands fluxes between warps through shared memory and recycles TMA ring slots behind a split barrier: a
    missed synchronisation would show as run-to-run differences.  30 launches on a many-tile, many-chunk grid and 5 on 256^3, on a
    side stream as well, all bit-identical to the first (which the tests above compare with the oracle)."""
    torch, wl = env["torch"], env["wl"]
    for dims, reps in (((264, 50, 36), 30), ((256, 256, 256), 5)):
        u = _field(dims, np.float32, 99, "noise")
        pr = wl.Projector(dims, np.float32)
        ud = torch.from_numpy(u).cuda()
        first = None
        side = torch.cuda.Stream()
        for it in range(reps):
            r = torch.full_like(ud, float("nan"))
            if it % 2:
                torch.cuda.synchronize()
                wl.wl_set_stream(pr.ctx, side)
            else:
                wl.wl_set_stream(pr.ctx, torch.cuda.current_stream())
            wl.wl_convdiff(pr.ctx, ud, 0.01, r)
            torch.cuda.synchronize()
            if first is None:
                first = r.clone()
                assert torch.isfinite(first).all()
            else:
                assert torch.equal(r.view(torch.int32), first.view(torch.int32)), (dims, it)
        wl.wl_set_stream(pr.ctx, torch.cuda.current_stream())
        pr.close()


def test_convdiff_misaligned_arrays_take_the_any_shape_kernel(env):
    """Caller arrays that do not start on a 16-byte boundary (a slice of a larger tensor) cannot be TMA sources: the call must
    fall back to the one-thread-per-cell kernel, not fail, and give the same field."""
    torch, wl = env["torch"], env["wl"]
    dims = (136, 24, 20)
    u = _field(dims, np.float32, 3, "smooth")
    ref = env["oracle"].convdiff(u, 0.02)
    pr = wl.Projector(dims, np.float32)
    n = u.size
    ubuf = torch.zeros(n + 4, dtype=torch.float32, device="cuda")
    rbuf = torch.full((n + 4,), float("nan"), dtype=torch.float32, device="cuda")
    ud = ubuf[1:1 + n].view(u.shape)
    rd = rbuf[3:3 + n].view(u.shape)
    assert ud.data_ptr() % 16 != 0 and rd.data_ptr() % 16 != 0
    ud.copy_(torch.from_numpy(u))
    wl.wl_convdiff(pr.ctx, ud, 0.02, rd)
    torch.cuda.synchronize()
    assert np.array_equal(rd.cpu().numpy(), ref)
    assert torch.isnan(rbuf[:3]).all() and torch.isnan(rbuf[3 + n:]).all()      # nothing written outside the field
    pr.close()


def test_convdiff_argument_errors(env):
    torch, wl = env["torch"], env["wl"]
    pr = wl.Projector((16, 8, 8), np.float32)
    u = pr.empty_faces()
    with pytest.raises(wl.WlError):
        wl.wl_convdiff(pr.ctx, u, 0.1, u)          # aliased
    pr.close()
