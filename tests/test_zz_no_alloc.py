"""wl_residual_norm_static — the one entry point of libwl.so that allocates nothing on the device.

It exists for the user who cannot call cudaMalloc where the residual check is needed: a solver whose fields already fill
the GPU, a plug-in inside a framework that owns all device memory through its own pool, a step loop that must not take
the device-wide stall of cudaMalloc / cudaFree.  The per-CTA partial sums, the running maximum and the CTA ticket live in a
fixed array inside the library image instead (about 128 KiB per GPU, grids up to WL_STATIC_MAX_CELLS = 2^27 cells).

Checked here: its output against the existing context path (wl_set_coeff + wl_residual_norm) within the tolerance the
other GPU tests use, on calls IN A ROW that share that array — the second with a different pressure field and then with a
smaller grid, so a maximum, ticket or partial left over from the call before would show; and that sizes beyond the limit
are refused before anything is launched.  The file sorts last on purpose (`pytest -x` stops at the first failure, and
this entry point lies outside the projection path): it passes alone in a fresh process and after the rest of the suite.
"""
import ctypes

import numpy as np
import pytest

RTOL = {np.float32: 1e-4, np.float64: 1e-10}   # BASELINE.json's bars, as in tests/test_gpu_path.py


def _fields(synth, config, scale, dt, seed):
    cfg = synth.make_config(config, dtype=dt, scale=scale)
    dims = cfg["dims"]
    shape = tuple(reversed(dims))
    M = int(np.prod(dims))
    L = cfg["L"].astype(dt)
    b = synth.uniform_pm1(seed, M, dtype=dt).reshape(shape)
    p = (synth.uniform_pm1(seed + 1, M, dtype=dt).reshape(shape) * dt(3.0) + dt(0.75)).astype(dt)   # non-zero mean
    return dims, L, p, b


@pytest.mark.gpu
@pytest.mark.parametrize("dt", [np.float32, np.float64])
def test_static_entry_matches_context_path_on_calls_in_a_row(dt):
    import torch
    from paper_2304_08159_b200 import binding as wl, build, synth
    build.build_cuda()
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    # (config, scale): 3-D 64^3 with a sphere (8 CTAs of the static kernel), then 2-D, then a small 3-D grid (1 CTA),
    # then the first grid again — each call inherits the scratch of the one before
    cases = [(2, 2, 11), (2, 2, 23), (1, 4, 31), (2, 8, 41), (2, 2, 11)]
    out = torch.full((2,), float("nan"), dtype=torch.float64, device="cuda")
    for config, scale, seed in cases:
        dims, L, p, b = _fields(synth, config, scale, dt, seed)
        Ld, pd, bd = (torch.from_numpy(a).cuda() for a in (L, p, b))
        # existing path: a context (allocates), its cleaned coefficient copy, three launches
        pr = wl.Projector(dims, dt)
        wl.wl_set_coeff(pr.ctx, Ld)
        r_ref, m_ref = wl.wl_residual_norm(pr.ctx, pd, bd)
        pr.close()
        # new path: no context, the caller's raw L, one launch, results left on the device
        out.fill_(float("nan"))
        assert wl.wl_residual_norm_static(dims, Ld, pd, bd, out) == wl.WL_OK
        torch.cuda.synchronize()
        r, m = out.cpu().numpy()
        assert np.isfinite(r) and np.isfinite(m), (dims, r, m)
        assert abs(r - r_ref) <= RTOL[dt] * r_ref, (dims, r, r_ref)
        assert abs(m - m_ref) <= RTOL[dt] * float(np.abs(p).max()), (dims, m, m_ref)
        assert abs(m - float(p.astype(np.float64).mean())) <= RTOL[dt] * float(np.abs(p).max())


@pytest.mark.gpu
def test_static_entry_two_calls_back_to_back_without_a_sync_between():
    """Two calls enqueued on one stream with no host synchronisation in between: stream order alone must keep the second
    call's clearing of the shared scratch behind the first call's kernel."""
    import torch
    from paper_2304_08159_b200 import binding as wl, build, synth
    build.build_cuda()
    dt = np.float32
    dims, L, p1, b = _fields(synth, 2, 2, dt, 7)
    p2 = (p1 * dt(-2.0) + dt(1.0)).astype(dt)
    Ld, bd, p1d, p2d = (torch.from_numpy(a).cuda() for a in (L, b, p1, p2))
    pr = wl.Projector(dims, dt)
    wl.wl_set_coeff(pr.ctx, Ld)
    ref1 = wl.wl_residual_norm(pr.ctx, p1d, bd)
    ref2 = wl.wl_residual_norm(pr.ctx, p2d, bd)
    pr.close()
    o1 = torch.zeros(2, dtype=torch.float64, device="cuda")
    o2 = torch.zeros(2, dtype=torch.float64, device="cuda")
    wl.wl_residual_norm_static(dims, Ld, p1d, bd, o1)
    wl.wl_residual_norm_static(dims, Ld, p2d, bd, o2)
    torch.cuda.synchronize()
    for got, ref, p in ((o1.cpu().numpy(), ref1, p1), (o2.cpu().numpy(), ref2, p2)):
        assert abs(got[0] - ref[0]) <= RTOL[dt] * ref[0], (got, ref)
        assert abs(got[1] - ref[1]) <= RTOL[dt] * float(np.abs(p).max()), (got, ref)


def test_static_entry_refuses_sizes_beyond_its_scratch():
    """The size check comes before any CUDA call, so it runs without a GPU too: nothing is dereferenced or launched."""
    from paper_2304_08159_b200 import binding as wl, build
    build.build_cuda()
    lib = wl.load()
    fake = ctypes.c_void_p(4096)          # never touched: the call must fail on the extents
    for dims in [(1024, 1024, 1024), (512, 512, 513), (16384, 16384)]:
        arr = (ctypes.c_int64 * 3)(*dims, *([1] * (3 - len(dims))))
        rc = lib.wl_residual_norm_static(len(dims), arr, wl.WL_F32, fake, fake, fake, fake, None)
        assert rc == wl.WL_EDIMS, (dims, rc)
        assert "WL_STATIC_MAX_CELLS" in wl.wl_static_last_error()
    ok = (ctypes.c_int64 * 3)(8, 8, 8)
    assert lib.wl_residual_norm_static(3, ok, wl.WL_F32, None, fake, fake, fake, None) == wl.WL_EINVAL
    assert lib.wl_residual_norm_static(3, ok, 5, fake, fake, fake, fake, None) == wl.WL_EINVAL
    assert lib.wl_residual_norm_static(3, ok, wl.WL_F32, fake, fake, fake, ctypes.c_void_p(4100), None) == wl.WL_EINVAL
    assert lib.wl_residual_norm_static(4, ok, wl.WL_F32, fake, fake, fake, fake, None) == wl.WL_EDIMS
    assert wl.WL_STATIC_MAX_CELLS == 512 ** 3
