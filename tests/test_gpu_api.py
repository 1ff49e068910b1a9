"""API behaviour on the GPU beyond plain parity: zero cycles, graph re-capture when the caller's buffers change, a
non-default stream, run-to-run determinism (a race in the fused kernels or the speculative enqueue would show here)."""
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


def _case(env, config=2, scale=2, dt=np.float32):
    torch, wl = env["torch"], env["wl"]
    cfg = env["synth"].make_config(config, dtype=dt, scale=scale)
    L, u = cfg["L"].astype(dt), cfg["u"].astype(dt)
    o = env["oracle"].Oracle(cfg["dims"], dt)
    o.set_coeff(L)
    b = o.divergence(u)
    pr = wl.Projector(cfg["dims"], dt)
    wl.wl_set_coeff(pr.ctx, torch.from_numpy(L).cuda())
    return cfg, o, b, pr


@pytest.mark.parametrize("config,scale", [(2, 2), (1, 4), (0, 1)])
def test_zero_cycles_returns_initial_residual_and_mean_free_p(env, config, scale):
    torch, wl = env["torch"], env["wl"]
    cfg, o, b, pr = _case(env, config, scale)
    rng = np.random.default_rng(5)
    p0 = rng.standard_normal(b.shape).astype(np.float32) + 3.0          # non-zero mean on purpose
    p_ref, hist_ref, nc_ref, rc_ref = o.solve(p0, b, 0.0, 0)
    p = torch.from_numpy(p0).cuda()
    hist, nc, rc = wl.wl_solve(pr.ctx, p, torch.from_numpy(b).cuda(), 0.0, 0)
    assert (nc, rc) == (nc_ref, rc_ref)
    assert hist.shape == (1,) and hist[0] == hist_ref[0]
    assert np.abs(p.cpu().numpy() - p_ref).max() <= 1e-6 * np.abs(p_ref).max()
    pr.close()


def test_new_buffers_recapture_the_graph(env):
    torch, wl = env["torch"], env["wl"]
    cfg, o, b, pr = _case(env)
    p_ref, hist_ref, _, _ = o.solve(np.zeros_like(b), b, 0.0, 5)
    for trial in range(3):                                             # fresh tensors each time: new pointers
        bd = torch.from_numpy(b.copy()).cuda()
        pad = torch.empty(1024 * (trial + 1), device="cuda")            # shift the allocator
        p = torch.zeros(b.shape, dtype=torch.float32, device="cuda")
        hist, nc, rc = wl.wl_solve(pr.ctx, p, bd, 0.0, 5)
        assert np.array_equal(hist, hist_ref)
        assert p.cpu().numpy().tobytes() == p_ref.tobytes()
        del pad
    pr.close()


def test_non_default_stream(env):
    torch, wl = env["torch"], env["wl"]
    cfg, o, b, pr = _case(env)
    p_ref, hist_ref, _, _ = o.solve(np.zeros_like(b), b, 0.0, 4)
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        wl.wl_set_stream(pr.ctx)                                        # the side stream (capturable directly)
        bd = torch.from_numpy(b).cuda()
        p = torch.zeros(b.shape, dtype=torch.float32, device="cuda")
        hist, nc, rc = wl.wl_solve(pr.ctx, p, bd, 0.0, 4)
        s.synchronize()
    assert np.array_equal(hist, hist_ref)
    assert p.cpu().numpy().tobytes() == p_ref.tobytes()
    pr.close()


@pytest.mark.parametrize("config,scale", [(4, 4), (1, 2)])
def test_repeated_solves_are_bit_reproducible(env, config, scale):
    torch, wl = env["torch"], env["wl"]
    cfg, o, b, pr = _case(env, config, scale)
    bd = torch.from_numpy(b).cuda()
    first = None
    for _ in range(5):
        p = torch.zeros(b.shape, dtype=torch.float32, device="cuda")
        hist, nc, rc = wl.wl_solve(pr.ctx, p, bd, 1e-4, 32)
        got = (p.cpu().numpy().tobytes(), hist.tobytes(), nc, rc)
        if first is None:
            first = got
        assert got == first
    pr.close()


def test_vcycle_call_matches_oracle_cycle(env):
    """wl_vcycle = one cycle + mean removal, norm of the returned p (the non-lagged path)."""
    torch, wl = env["torch"], env["wl"]
    cfg, o, b, pr = _case(env)
    bd = torch.from_numpy(b).cuda()
    p = torch.zeros(b.shape, dtype=torch.float32, device="cuda")
    p_ref = np.zeros_like(b)
    for _ in range(3):
        nrm = wl.wl_vcycle(pr.ctx, p, bd)
        p_ref, nrm_ref = o.vcycle(p_ref, b)
        assert nrm == nrm_ref
    assert p.cpu().numpy().tobytes() == p_ref.tobytes()
    pr.close()


@pytest.mark.parametrize("config,scale", [(2, 2), (1, 4)])
def test_solve_kernels_option_does_not_leak_into_the_solvers(env, config, scale):
    """WL_OPT_SOLVE_KERNELS is a profiling switch of the wl_down / wl_up entry points.  With it set (and the solve history
    allocated by an earlier solve) wl_vcycle, the plain wl_solve and wl_solve_pcg must still run their own kernel instances:
    the solve instances subtract a stale mean on load and bump the cycle counter."""
    torch, wl = env["torch"], env["wl"]
    cfg, o, b, pr = _case(env, config, scale)
    bd = torch.from_numpy(b).cuda()
    p = torch.zeros(b.shape, dtype=torch.float32, device="cuda")
    wl.wl_solve(pr.ctx, p, bd, 0.0, 3)                                   # allocates the history, leaves a non-zero shift behind
    wl.wl_set_option(pr.ctx, wl.WL_OPT_SOLVE_KERNELS, 1)
    p0 = np.random.default_rng(9).standard_normal(b.shape).astype(np.float32) + np.float32(2.0)
    p_ref, r_ref = o.vcycle(p0, b)
    p1 = torch.from_numpy(p0).cuda()
    r1 = wl.wl_vcycle(pr.ctx, p1, bd)
    assert np.abs(p1.cpu().numpy() - p_ref).max() <= 1e-4 * np.abs(p_ref).max()
    assert abs(r1 / r_ref - 1) <= 1e-3
    wl.wl_set_option(pr.ctx, wl.WL_OPT_GRAPH, 0)                         # the non-lagged, non-graph solve calls down()/up() too
    for solver, ref in ((wl.wl_solve, o.solve), (wl.wl_solve_pcg, o.solve_pcg)):
        p_ref, hist_ref, nc_ref, rc_ref = ref(np.zeros_like(b), b, 0.0, 4)
        p2 = torch.zeros(b.shape, dtype=torch.float32, device="cuda")
        hist, nc, rc = solver(pr.ctx, p2, bd, 0.0, 4)
        assert (nc, rc) == (nc_ref, rc_ref)
        assert np.abs(hist / hist_ref - 1).max() <= 1e-3, (hist, hist_ref)
        assert np.abs(p2.cpu().numpy() - p_ref).max() <= 1e-4 * np.abs(p_ref).max()
    pr.close()
