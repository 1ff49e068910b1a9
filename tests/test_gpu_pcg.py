"""T2 — parity of wl_solve_pcg (V-cycle-preconditioned conjugate gradients) against
the oracle's solve_pcg (pinned by tests/test_oracle_pcg.py).  Bars as for wl_solve (BASELINE.json "Numerical agreement"):
fp32 p within 1e-4 max|p_cpu|, every hist[k] within 1e-3; fp64 1e-10.  The GPU sums its dot products in another order
than the oracle (fp64 partials per CTA, ordered second stage): alpha and beta agree to ~1e-16 before the cast to T, so
fp32 iterates are normally bit-identical as well (reported, not required)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

P_TOL = {np.dtype(np.float32): 1e-4, np.dtype(np.float64): 1e-10}
H_TOL = {np.dtype(np.float32): 1e-3, np.dtype(np.float64): 1e-10}


@pytest.fixture(scope="module")
def env(oracle_mod):
    import torch
    from paper_2304_08159_b200 import binding as wl, build, synth
    build.build_cuda()
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return dict(torch=torch, wl=wl, oracle=oracle_mod, synth=synth)


def _setup(env, cfg, dt, fused=1, graph=1):
    torch, wl = env["torch"], env["wl"]
    o = env["oracle"].Oracle(cfg["dims"], dt)
    L, u = cfg["L"].astype(dt), cfg["u"].astype(dt)
    o.set_coeff(L)
    b = o.divergence(u)
    pr = wl.Projector(cfg["dims"], dt)
    wl.wl_set_option(pr.ctx, wl.WL_OPT_FUSED, fused)
    wl.wl_set_option(pr.ctx, wl.WL_OPT_GRAPH, graph)
    wl.wl_set_coeff(pr.ctx, torch.from_numpy(L).cuda())
    return o, b, pr


def _compare(p, p_ref, hist, hist_ref, dt):
    assert hist.shape == hist_ref.shape, (hist, hist_ref)
    assert np.abs(hist / hist_ref - 1.0).max() <= H_TOL[np.dtype(dt)], (hist, hist_ref)
    err = np.abs(p.astype(np.float64) - p_ref.astype(np.float64)).max() / np.abs(p_ref).max()
    assert err <= P_TOL[np.dtype(dt)], err


@pytest.mark.parametrize("config,scale,dt", [(0, 1, np.float32), (1, 4, np.float32), (1, 4, np.float64), (2, 2, np.float32),
                                             (2, 2, np.float64), (3, 4, np.float32), (4, 4, np.float32), (4, 8, np.float64)])
@pytest.mark.parametrize("fused,graph", [(0, 0), (1, 1)])
def test_fixed_iteration_count(env, config, scale, dt, fused, graph):
    """Exactly K iterations (tol = 0) on both sides."""
    torch, wl = env["torch"], env["wl"]
    cfg = env["synth"].make_config(config, dtype=dt, scale=scale)
    o, b, pr = _setup(env, cfg, dt, fused, graph)
    K = 6
    p_ref, hist_ref, nit_ref, rc_ref = o.solve_pcg(np.zeros_like(b), b, 0.0, K)
    p = pr.zeros_cells()
    hist, nit, rc = wl.wl_solve_pcg(pr.ctx, p, torch.from_numpy(b).cuda(), 0.0, K)
    assert (nit, rc) == (nit_ref, rc_ref) == (K, wl.WL_NOT_CONVERGED)
    _compare(p.cpu().numpy(), p_ref, hist, hist_ref, dt)
    assert abs(p.double().mean().item()) <= 10 * np.finfo(dt).eps * np.abs(p_ref).max()
    pr.close()


@pytest.mark.parametrize("config,scale", [(1, 2), (2, 1), (3, 2), (4, 4)])
def test_to_tolerance_and_fewer_cycles_than_plain_cycling(env, config, scale):
    """Solve to 1e-4·||b||inf: same iteration count, history and p as the oracle; fewer V-cycles than wl_solve needs."""
    torch, wl = env["torch"], env["wl"]
    dt = np.float32
    cfg = env["synth"].make_config(config, dtype=dt, scale=scale)
    o, b, pr = _setup(env, cfg, dt)
    p_ref, hist_ref, nit_ref, rc_ref = o.solve_pcg(np.zeros_like(b), b, 1e-4, 32)
    bd = torch.from_numpy(b).cuda()
    p = pr.zeros_cells()
    hist, nit, rc = wl.wl_solve_pcg(pr.ctx, p, bd, 1e-4, 32)
    assert (nit, rc) == (nit_ref, rc_ref), (hist, hist_ref)
    assert rc == 0
    _compare(p.cpu().numpy(), p_ref, hist, hist_ref, dt)
    _, rtrue = o.residual(p.cpu().numpy(), b)
    assert rtrue <= 1.1e-4 * np.abs(b).max()                      # the recurrence residual tracks the true one
    p2 = pr.zeros_cells()
    hist2, nc2, rc2 = wl.wl_solve(pr.ctx, p2, bd, 1e-4, 64)
    assert nit < nc2
    # repeat call through the cached graph, warm start from the solution: zero iterations
    hist3, nit3, rc3 = wl.wl_solve_pcg(pr.ctx, p, bd, 2e-4, 32)
    assert nit3 == 0 and rc3 == 0
    pr.close()


def test_project_with_the_cg_solver(env):
    """wl_project with WL_OPT_SOLVER = 1: divergence, PCG solve, gradient correction — against the oracle's pieces."""
    torch, wl = env["torch"], env["wl"]
    dt = np.float32
    cfg = env["synth"].make_config(2, dtype=dt, scale=2)
    o, b, pr = _setup(env, cfg, dt)
    wl.wl_set_option(pr.ctx, wl.WL_OPT_SOLVER, 1)
    p_ref, hist_ref, nit_ref, rc_ref = o.solve_pcg(np.zeros_like(b), b, 1e-4, 32)
    u_ref = o.gradient_correct(cfg["u"], p_ref)
    ud = torch.from_numpy(cfg["u"]).cuda()
    p = pr.zeros_cells()
    hist, nit, rc = wl.wl_project(pr.ctx, ud, None, p, 1e-4, 32)
    assert (nit, rc) == (nit_ref, rc_ref)
    _compare(p.cpu().numpy(), p_ref, hist, hist_ref, dt)
    assert np.abs(ud.cpu().numpy() - u_ref).max() <= 1e-4 * np.abs(u_ref).max()
    assert np.abs(o.divergence(ud.cpu().numpy())).max() <= 1.1e-4 * hist[0]
    pr.close()


def test_zero_right_hand_side_stops_at_once(env):
    torch, wl = env["torch"], env["wl"]
    cfg = env["synth"].make_config(2, scale=4)
    o, b, pr = _setup(env, cfg, np.float32)
    p = torch.full(pr.cell_shape(), 2.5, dtype=torch.float32, device="cuda")
    hist, nit, rc = wl.wl_solve_pcg(pr.ctx, p, torch.zeros_like(p), 1e-4, 8)
    assert nit == 0 and rc == 0 and hist[0] == 0.0 and p.abs().max().item() == 0.0
    pr.close()
