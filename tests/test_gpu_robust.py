"""Robustness of the C ABI on the GPU: non-finite input is reported instead of reading as "converged";
16-byte-misaligned caller arrays fall back to the generic kernels instead of failing in the tensor-map encoder; a time
stepper alternating two pressure buffers does not re-capture its V-cycle graph on every call."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def env(oracle_mod):
    import torch
    from paper_2304_08159_b200 import binding as wl, build, synth
    build.build_cuda()
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return dict(torch=torch, wl=wl, oracle=oracle_mod, synth=synth)


@pytest.mark.parametrize("config,scale", [(2, 2), (1, 4)])
@pytest.mark.parametrize("where", ["b", "p"])
def test_non_finite_input_is_reported(env, config, scale, where):
    torch, wl = env["torch"], env["wl"]
    cfg = env["synth"].make_config(config, scale=scale)
    pr = wl.Projector(cfg["dims"], np.float32)
    wl.wl_set_coeff(pr.ctx, torch.from_numpy(cfg["L"]).cuda())
    b = pr.empty_cells()
    wl.wl_divergence(pr.ctx, torch.from_numpy(cfg["u"]).cuda(), b)
    p = pr.zeros_cells()
    idx = tuple(s // 2 + 1 for s in p.shape)
    (b if where == "b" else p)[idx] = float("nan")
    for fn in (wl.wl_solve, wl.wl_solve_pcg):
        with pytest.raises(wl.WlError) as ei:
            fn(pr.ctx, p.clone(), b, 1e-4, 8)
        assert ei.value.code == wl.WL_ENONFINITE
    pr.close()


@pytest.mark.parametrize("dims", [(64, 48, 32), (128, 64)])
def test_misaligned_caller_arrays_fall_back_to_the_generic_kernels(env, dims):
    torch, wl, o = env["torch"], env["wl"], env["oracle"]
    dt = np.float32
    rng = np.random.default_rng(3)
    n = len(dims)
    shape = tuple(reversed(dims))
    L = env["synth"].coeff_uniform(dims, dt)
    u = (rng.uniform(-1, 1, size=(n,) + shape).astype(dt) * L).astype(dt)
    orc = o.Oracle(dims, dt)
    orc.set_coeff(L)
    b = orc.divergence(u)
    p_ref, hist_ref, nc_ref, rc_ref = orc.solve(np.zeros(shape, dt), b, 0.0, 4)
    pr = wl.Projector(dims, dt)
    wl.wl_set_coeff(pr.ctx, torch.from_numpy(L).cuda())
    M = int(np.prod(dims))
    raw_p = torch.zeros(M + 4, dtype=torch.float32, device="cuda")
    raw_b = torch.zeros(M + 4, dtype=torch.float32, device="cuda")
    p = raw_p[1:M + 1].view(shape)                                    # 4 bytes off a 16-byte boundary
    bd = raw_b[1:M + 1].view(shape)
    assert p.data_ptr() % 16 == 4 and p.is_contiguous()
    bd.copy_(torch.from_numpy(b))
    hist, nc, rc = wl.wl_solve(pr.ctx, p, bd, 0.0, 4)
    assert nc == nc_ref
    assert np.abs(hist / hist_ref - 1.0).max() <= 1e-3
    assert np.abs(p.cpu().numpy() - p_ref).max() <= 1e-4 * np.abs(p_ref).max()
    pr.close()


def test_alternating_buffers_reuse_their_graphs(env):
    torch, wl = env["torch"], env["wl"]
    cfg = env["synth"].make_config(2, scale=4)
    pr = wl.Projector(cfg["dims"], np.float32)
    wl.wl_set_coeff(pr.ctx, torch.from_numpy(cfg["L"]).cuda())
    b = pr.empty_cells()
    wl.wl_divergence(pr.ctx, torch.from_numpy(cfg["u"]).cuda(), b)
    pa, pb = pr.zeros_cells(), pr.zeros_cells()
    ha, _, _ = wl.wl_solve(pr.ctx, pa, b, 0.0, 3)
    hb, _, _ = wl.wl_solve(pr.ctx, pb, b, 0.0, 3)
    assert np.array_equal(ha, hb)
    import time
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(10):                                                # both graphs stay cached: no re-capture
        pa.zero_(); pb.zero_()
        h1, _, _ = wl.wl_solve(pr.ctx, pa, b, 0.0, 3)
        h2, _, _ = wl.wl_solve(pr.ctx, pb, b, 0.0, 3)
        assert np.array_equal(h1, ha) and np.array_equal(h2, ha)
    torch.cuda.synchronize()
    per_call = (time.perf_counter() - t0) / 20
    assert per_call < 5e-3, per_call                                  # a re-capture + instantiate costs milliseconds
    assert torch.equal(pa, pb)
    pr.close()
