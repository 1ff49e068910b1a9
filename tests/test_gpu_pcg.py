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


@pytest.mark.parametrize("fused,graph", [(0, 0), (1, 1)])
def test_breakdown_then_recover(env, fused, graph):
    """An all-solid field (L = 0: A = 0, D = 0, so z = V(r) = 0 and r·z = 0) breaks the iteration down at once; the oracle
    returns p untouched but for the mean, nit = 0 and — since hist[0] = ||b||inf is above the tolerance — rc 1.  The next
    solve on the same context, after wl_set_coeff installed a valid field, must not inherit the breakdown flag."""
    torch, wl = env["torch"], env["wl"]
    dt = np.float32
    cfg = env["synth"].make_config(2, dtype=dt, scale=4)
    o, b, pr = _setup(env, cfg, dt, fused, graph)
    bd = torch.from_numpy(b).cuda()
    L0 = np.zeros_like(cfg["L"])
    o.set_coeff(L0)
    wl.wl_set_coeff(pr.ctx, torch.from_numpy(L0).cuda())
    rng = np.random.default_rng(3)
    p0 = rng.standard_normal(b.shape).astype(dt) + dt(0.5)
    p_ref, hist_ref, nit_ref, rc_ref = o.solve_pcg(p0, b, 1e-4, 8)
    assert (nit_ref, rc_ref) == (0, 1) and hist_ref[0] == np.abs(b).max()
    p = torch.from_numpy(p0).cuda()
    hist, nit, rc = wl.wl_solve_pcg(pr.ctx, p, bd, 1e-4, 8)
    assert (nit, rc) == (nit_ref, rc_ref), (hist, nit, rc)
    assert np.array_equal(hist, hist_ref)
    assert np.abs(p.cpu().numpy() - p_ref).max() <= 1e-6 * np.abs(p_ref).max()
    # recover: valid coefficients, same context
    L = cfg["L"].astype(dt)
    o.set_coeff(L)
    wl.wl_set_coeff(pr.ctx, torch.from_numpy(L).cuda())
    p_ref, hist_ref, nit_ref, rc_ref = o.solve_pcg(np.zeros_like(b), b, 1e-4, 32)
    assert nit_ref > 0 and rc_ref == 0
    p = pr.zeros_cells()
    hist, nit, rc = wl.wl_solve_pcg(pr.ctx, p, bd, 1e-4, 32)
    assert (nit, rc) == (nit_ref, rc_ref), (hist, hist_ref)
    _compare(p.cpu().numpy(), p_ref, hist, hist_ref, dt)
    # and through wl_project with the CG solver selected
    wl.wl_set_option(pr.ctx, wl.WL_OPT_SOLVER, 1)
    ud = torch.from_numpy(cfg["u"].astype(dt)).cuda()
    p2 = pr.zeros_cells()
    hist2, nit2, rc2 = wl.wl_project(pr.ctx, ud, None, p2, 1e-4, 32)
    assert (nit2, rc2) == (nit_ref, rc_ref)
    pr.close()


@pytest.mark.parametrize("opt,val", [("WL_OPT_PDL", 0), ("WL_OPT_COARSE_CTA", 0)])
@pytest.mark.parametrize("config,scale", [(2, 2), (1, 4)])
def test_pdl_and_coarse_tail_off_give_the_same_bits(env, config, scale, opt, val):
    """Programmatic dependent launch only overlaps a kernel's prologue with its predecessor's drain, and the single-CTA coarse
    tail does the arithmetic of the per-level kernels: switching either off must not change one bit of p or of the history,
    for wl_solve and for wl_solve_pcg (a read ahead of griddepcontrol.wait would show here)."""
    torch, wl = env["torch"], env["wl"]
    dt = np.float32
    cfg = env["synth"].make_config(config, dtype=dt, scale=scale)
    res = {}
    for setting in (1, val):
        o, b, pr = _setup(env, cfg, dt)
        wl.wl_set_option(pr.ctx, getattr(wl, opt), setting)
        bd = torch.from_numpy(b).cuda()
        p = pr.zeros_cells()
        h1, n1, _ = wl.wl_solve(pr.ctx, p, bd, 0.0, 5)
        q = pr.zeros_cells()
        h2, n2, _ = wl.wl_solve_pcg(pr.ctx, q, bd, 0.0, 5)
        res[setting] = (p.clone(), h1, q.clone(), h2)
        pr.close()
    a, c = res[1], res[val]
    assert torch.equal(a[0], c[0]) and np.array_equal(a[1], c[1])
    assert torch.equal(a[2], c[2]) and np.array_equal(a[3], c[3])
    p_ref, hist_ref, _, _ = o.solve_pcg(np.zeros_like(b), b, 0.0, 5)
    _compare(c[2].cpu().numpy(), p_ref, c[3], hist_ref, dt)


def test_misaligned_x_takes_the_scalar_update_kernels(env):
    """p handed in as a torch slice that starts 4 bytes off a 16-byte boundary: level 0 falls back to the generic kernels and
    the vector updates to their scalar forms; the result must still be the oracle's."""
    torch, wl = env["torch"], env["wl"]
    dt = np.float32
    cfg = env["synth"].make_config(2, dtype=dt, scale=4)
    o, b, pr = _setup(env, cfg, dt)
    M = int(np.prod(cfg["dims"]))
    store = torch.zeros(M + 8, dtype=torch.float32, device="cuda")
    off = 1 if store.data_ptr() % 16 == 0 else 0
    p = store[off + 0: off + M].view(pr.cell_shape())
    assert p.data_ptr() % 16 != 0 and p.is_contiguous()
    p_ref, hist_ref, nit_ref, rc_ref = o.solve_pcg(np.zeros_like(b), b, 0.0, 5)
    hist, nit, rc = wl.wl_solve_pcg(pr.ctx, p, torch.from_numpy(b).cuda(), 0.0, 5)
    assert (nit, rc) == (nit_ref, rc_ref)
    _compare(p.cpu().numpy(), p_ref, hist, hist_ref, dt)
    pr.close()


@pytest.mark.parametrize("config,dt", [(3, np.float32), (3, np.float64), (4, np.float32)])
def test_full_size_six_iterations(env, config, dt, capsys):
    """BASELINE configs[3] (256^3, fp32 and fp64) and configs[4] (512^3 fp32, 32 spheres) at FULL size, K = 6 iterations
    (tol = 0) through the launch configuration bench.py's `pcg` leg reports: 144/148-CTA level-0 plans, the UP kernel that also
    sums r·z over its per-CTA partials, one graph launch per iteration.  p element-wise and hist[0..6] against oracle.solve_pcg
    at BASELINE.json's bars (the twin of test_config4_full_512_eight_cycles).  The fp32
    bit-identity with the oracle is reported, not required (the dot products are summed in another order)."""
    torch, wl = env["torch"], env["wl"]
    cfg = env["synth"].make_config(config, dtype=dt)
    o, b, pr = _setup(env, cfg, dt)
    K = 6
    p_ref, hist_ref, nit_ref, rc_ref = o.solve_pcg(np.zeros_like(b), b, 0.0, K)
    p = pr.zeros_cells()
    hist, nit, rc = wl.wl_solve_pcg(pr.ctx, p, torch.from_numpy(b).cuda(), 0.0, K)
    assert (nit, rc) == (nit_ref, rc_ref) == (K, wl.WL_NOT_CONVERGED)
    pg = p.cpu().numpy()
    _compare(pg, p_ref, hist, hist_ref, dt)
    assert hist.shape == (K + 1,) and hist[-1] < 1e-2 * hist[0]
    with capsys.disabled():
        print(f"\n[pcg full size] {cfg['name']} {np.dtype(dt).name}: p bit-identical={pg.tobytes() == p_ref.tobytes()} "
              f"hist bit-identical={np.array_equal(hist, hist_ref)} max rel hist dev={np.abs(hist / hist_ref - 1).max():.2e}")
    pr.close()
