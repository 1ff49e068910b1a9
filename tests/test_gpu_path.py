"""T2 — path parity of wl_vcycle / wl_solve / wl_project against the oracle on the BASELINE.json configs.

Bars (BASELINE.json north_star "Numerical agreement"):
  fp32: max|p_gpu - p_cpu| <= 1e-4 max|p_cpu| after a fixed cycle count; every per-cycle ||r||inf within 1e-3 relative;
  fp64: 1e-10 for both.  Cycle counts to tolerance must be equal (+-1 only if the oracle's stopping residual is within
  1e-3 relative of tol·||b||, i.e. the stop decision itself is inside the parity tolerance).
Full sizes use the launch configuration bench.py times (fused kernels + CUDA graph + lagged stop test = the defaults of
wl_solve / wl_project): K = 8 cycles of wl_solve(tol = 0) are compared element by element (p) and cycle by cycle (hist)
with the oracle at 256^3 fp32 / fp64 and 512^3 fp32 (the oracle needs ~8 s per 512^3 V-cycle), and
the converged 512^3 projection is checked in addition by properties the oracle evaluates on the GPU's own output.
"""
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


def _projector(env, cfg, dt, fused=1, graph=1):
    wl = env["wl"]
    pr = wl.Projector(cfg["dims"], dt)
    wl.wl_set_option(pr.ctx, wl.WL_OPT_FUSED, fused)
    wl.wl_set_option(pr.ctx, wl.WL_OPT_GRAPH, graph)
    return pr


def _check_hist(hist, ref, dt):
    assert hist.shape == ref.shape, (hist.shape, ref.shape)
    rel = np.abs(hist / ref - 1.0).max()
    assert rel <= H_TOL[np.dtype(dt)], (rel, hist, ref)


def _check_p(p, ref, dt):
    err = np.abs(p.astype(np.float64) - ref.astype(np.float64)).max() / np.abs(ref).max()
    assert err <= P_TOL[np.dtype(dt)], err
    return err


def _run_solve_parity(env, cfg, dt, K, fused=1, graph=1, bitwise=False):
    """Exactly K cycles (tol = 0) on both sides; p and history compared.  bitwise: also the fp32 drift alarm (p and hist
    bit-identical to the oracle's: DESIGN.md §3 reading 12)."""
    torch, wl = env["torch"], env["wl"]
    o = env["oracle"].Oracle(cfg["dims"], dt)
    L, u = cfg["L"].astype(dt), cfg["u"].astype(dt)
    o.set_coeff(L)
    b = o.divergence(u)
    p_ref, hist_ref, nc_ref, rc_ref = o.solve(np.zeros_like(b), b, 0.0, K)
    pr = _projector(env, cfg, dt, fused, graph)
    wl.wl_set_coeff(pr.ctx, torch.from_numpy(L).cuda())
    bd = pr.empty_cells()
    wl.wl_divergence(pr.ctx, torch.from_numpy(u).cuda(), bd)
    p = pr.zeros_cells()
    hist, nc, rc = wl.wl_solve(pr.ctx, p, bd, 0.0, K)
    assert (nc, rc) == (nc_ref, rc_ref) == (K, wl.WL_NOT_CONVERGED)
    _check_hist(hist, hist_ref, dt)
    pg = p.cpu().numpy()
    _check_p(pg, p_ref, dt)
    assert abs(p.double().mean().item()) <= 10 * np.finfo(dt).eps * np.abs(p_ref).max()
    if bitwise:
        assert np.array_equal(hist, hist_ref), np.abs(hist / hist_ref - 1).max()
        assert pg.tobytes() == p_ref.tobytes()
    pr.close()
    return hist_ref


@pytest.mark.parametrize("fused,graph", [(0, 0), (1, 0), (1, 1)])
def test_config0_ten_cycles(env, fused, graph):
    """BASELINE configs[0]: 2-D 64x64 fp32 uniform, 4 coarsenings, 10 V-cycles, p0 = 0."""
    cfg = env["synth"].make_config(0)
    hist = _run_solve_parity(env, cfg, np.float32, 10, fused, graph)
    assert hist.shape == (11,)


@pytest.mark.parametrize("config,scale,dt", [(1, 4, np.float32), (1, 4, np.float64), (2, 2, np.float32),
                                             (2, 2, np.float64), (3, 4, np.float32), (3, 4, np.float64),
                                             (4, 4, np.float32)])
@pytest.mark.parametrize("fused,graph", [(0, 0), (1, 1)])
def test_reduced_configs_fixed_cycles(env, config, scale, dt, fused, graph):
    cfg = env["synth"].make_config(config, dtype=dt, scale=scale)
    _run_solve_parity(env, cfg, dt, 8, fused, graph)


def _run_to_tolerance(env, cfg, dt, fused=1, graph=1):
    torch, wl = env["torch"], env["wl"]
    o = env["oracle"].Oracle(cfg["dims"], dt)
    L, u = cfg["L"].astype(dt), cfg["u"].astype(dt)
    shape = tuple(reversed(cfg["dims"]))
    pr = _projector(env, cfg, dt, fused, graph)
    ud = torch.from_numpy(u).cuda()
    Ld = torch.from_numpy(L).cuda()
    p = pr.zeros_cells()
    if cfg["call"] == "project":
        u_ref, p_ref, hist_ref, nc_ref, rc_ref = o.project(u, L, np.zeros(shape, dt), cfg["tol"], cfg["maxcycles"])
        hist, nc, rc = wl.wl_project(pr.ctx, ud, Ld, p, cfg["tol"], cfg["maxcycles"])
    else:
        o.set_coeff(L)
        b = o.divergence(u)
        p_ref, hist_ref, nc_ref, rc_ref = o.solve(np.zeros(shape, dt), b, cfg["tol"], cfg["maxcycles"])
        wl.wl_set_coeff(pr.ctx, Ld)
        bd = pr.empty_cells()
        wl.wl_divergence(pr.ctx, ud, bd)
        hist, nc, rc = wl.wl_solve(pr.ctx, p, bd, cfg["tol"], cfg["maxcycles"])
        u_ref = None
    if nc != nc_ref:
        # allowed only when the stop decision is inside the parity tolerance (c-20)
        thr = cfg["tol"] * hist_ref[0]
        k = min(nc, nc_ref)
        assert abs(nc - nc_ref) == 1 and abs(hist_ref[k] / thr - 1.0) <= H_TOL[np.dtype(dt)], (nc, nc_ref, hist, hist_ref)
    else:
        assert rc == rc_ref
        _check_hist(hist, hist_ref, dt)
        _check_p(p.cpu().numpy(), p_ref, dt)
        if u_ref is not None:
            du = np.abs(ud.cpu().numpy() - u_ref).max() / np.abs(u_ref).max()
            assert du <= P_TOL[np.dtype(dt)], du
    pr.close()
    return nc, rc


def test_config1_full_cylinder_to_tolerance(env):
    """BASELINE configs[1]: 2-D 1024x1024 fp32 cylinder, solve to 1e-4 (expected to end at the 32-cycle cap; c-19)."""
    cfg = env["synth"].make_config(1)
    nc, rc = _run_to_tolerance(env, cfg, np.float32)
    assert nc >= 20


def test_config2_full_sphere_project(env):
    """BASELINE configs[2]: 3-D 128^3 fp32 sphere, full wl_project."""
    cfg = env["synth"].make_config(2)
    nc, rc = _run_to_tolerance(env, cfg, np.float32)
    assert rc == 0 and 10 <= nc <= 32


@pytest.mark.parametrize("dt", [np.float32, np.float64])
def test_config3_full_256_eight_cycles(env, dt):
    """BASELINE configs[3]: 3-D 256^3 uniform L, Taylor-Green + noise, fp32 and fp64 (6 coarsenings): K = 8 cycles of the
    lagged, graph-launched wl_solve (what bench.py times) against oracle.solve, p element-wise and hist[0..8] (c-20)."""
    cfg = env["synth"].make_config(3, dtype=dt)
    hist = _run_solve_parity(env, cfg, dt, 8, bitwise=(dt == np.float32))
    assert hist.shape == (9,)


def test_config4_full_512_eight_cycles(env):
    """BASELINE configs[4] at FULL size through the entry point and launch configuration bench.py times (wl_solve:
    fused level halves, one CUDA graph per cycle, lagged device-side stop test): K = 8 cycles, p element-wise within
    1e-4 max|p_cpu|, hist[0..8] within 1e-3 (c-20, c-21), plus the fp32 bit-identity drift alarm."""
    cfg = env["synth"].make_config(4)
    hist = _run_solve_parity(env, cfg, np.float32, 8, bitwise=True)
    assert hist.shape == (9,) and np.all(np.diff(hist) < 0)


def test_config3_half_size_to_tolerance_fp64(env):
    cfg = env["synth"].make_config(3, dtype=np.float64, scale=2)
    nc, rc = _run_to_tolerance(env, cfg, np.float64)
    assert rc == 0


def test_config4_full_512_properties_and_two_cycles(env):
    """BASELINE configs[4]: 3-D 512^3 fp32, 32 spheres, wl_project to tolerance — bench.py's workload and launch
    configuration.  The oracle needs 17 s per V-cycle here, so: (a) two V-cycles compared element by element;
    (b) the converged projection checked by what the ORACLE computes from the GPU's own p and u:
    hist[-1] = ||b - A p||inf, div(u_out) = b - A p, u_out = u - L grad p, mean(p) = 0, monotone history."""
    torch, wl = env["torch"], env["wl"]
    dt = np.float32
    cfg = env["synth"].make_config(4)
    L, u = cfg["L"], cfg["u"]
    o = env["oracle"].Oracle(cfg["dims"], dt)
    o.set_coeff(L)
    b = o.divergence(u)
    pr = _projector(env, cfg, dt)
    Ld = torch.from_numpy(L).cuda()
    ud = torch.from_numpy(u).cuda()
    wl.wl_set_coeff(pr.ctx, Ld)
    bd = pr.empty_cells()
    wl.wl_divergence(pr.ctx, ud, bd)
    assert np.abs(bd.cpu().numpy() - b).max() <= 1e-6
    # (a) two cycles
    p = pr.zeros_cells()
    p_ref = np.zeros_like(b)
    for k in range(2):
        nrm = wl.wl_vcycle(pr.ctx, p, bd)
        p_ref, nrm_ref = o.vcycle(p_ref, b)
        assert abs(nrm / nrm_ref - 1.0) <= 1e-3
    _check_p(p.cpu().numpy(), p_ref, dt)
    del p_ref
    # (b) full projection
    p.zero_()
    hist, nc, rc = wl.wl_project(pr.ctx, ud, None, p, cfg["tol"], cfg["maxcycles"])
    assert rc == 0 and 10 <= nc <= 32
    assert np.all(np.diff(hist) < 0)
    assert hist[0] == np.abs(b).max()
    assert hist[-1] <= cfg["tol"] * hist[0] < hist[-2]
    pg = p.cpu().numpy()
    r, nrm = o.residual(pg, b)
    assert abs(hist[-1] / nrm - 1.0) <= 1e-3
    assert abs(pg.astype(np.float64).mean()) <= 1e-6 * np.abs(pg).max()
    ug = ud.cpu().numpy()
    u_exp = o.gradient_correct(u, pg)
    assert np.abs(ug - u_exp).max() <= 1e-6 * max(1.0, np.abs(u_exp).max())
    div_after = o.divergence(ug)
    assert np.abs(div_after).max() <= 1.1e-4 * hist[0]
    assert np.abs(div_after - r).max() <= 2e-5 * hist[0]
    pr.close()


def test_warm_start_and_repeat_calls(env):
    """Projecting the already-corrected field starts from a divergence that is the first call's final residual; solving
    again from the solution runs zero cycles and leaves p unchanged up to its (already zero) mean."""
    torch, wl = env["torch"], env["wl"]
    cfg = env["synth"].make_config(2, scale=4)
    pr = _projector(env, cfg, np.float32)
    ud = torch.from_numpy(cfg["u"]).cuda()
    bd = pr.empty_cells()
    wl.wl_divergence(pr.ctx, ud, bd)
    p = pr.zeros_cells()
    hist, nc, rc = wl.wl_project(pr.ctx, ud, torch.from_numpy(cfg["L"]).cuda(), p, 1e-4, 32)
    assert rc == 0 and nc > 5
    b2 = pr.empty_cells()
    wl.wl_divergence(pr.ctx, ud, b2)
    assert abs(b2.abs().max().item() / hist[-1] - 1.0) <= 1e-3   # div(u_out) = b - A p
    p_before = p.clone()
    hist2, nc2, rc2 = wl.wl_solve(pr.ctx, p, bd, 1e-4, 32)
    assert nc2 == 0 and rc2 == 0 and hist2.shape == (1,) and abs(hist2[0] / hist[-1] - 1.0) <= 1e-3
    assert (p - p_before).abs().max().item() <= 1e-6 * p_before.abs().max().item()
    pr.close()


def test_project_host_matches_device_call(env):
    torch, wl = env["torch"], env["wl"]
    cfg = env["synth"].make_config(2, scale=4)
    pr = _projector(env, cfg, np.float32)
    ud = torch.from_numpy(cfg["u"]).cuda()
    Ld = torch.from_numpy(cfg["L"]).cuda()
    p = pr.zeros_cells()
    hist, nc, rc = wl.wl_project(pr.ctx, ud, Ld, p, 1e-4, 32)
    uh = torch.from_numpy(cfg["u"].copy()).pin_memory()
    Lh = torch.from_numpy(cfg["L"].copy()).pin_memory()
    ph = torch.zeros(pr.cell_shape(), dtype=torch.float32).pin_memory()
    hist_h, nc_h, rc_h = wl.wl_project_host(pr.ctx, uh, Lh, ph, 1e-4, 32)
    assert nc_h == nc and rc_h == rc and np.array_equal(hist_h, hist)
    assert torch.equal(uh, ud.cpu()) and torch.equal(ph, p.cpu())
    pr.close()


@pytest.mark.parametrize("config,scale,dt,K", [(0, 1, np.float32, 10), (1, 4, np.float32, 12), (2, 2, np.float32, 8),
                                                (3, 4, np.float32, 6), (4, 8, np.float32, 8)])
def test_bit_identical_iterates_and_history(env, config, scale, dt, K):
    """Drift alarm, beyond BASELINE's tolerances: the library is compiled without FMA contraction and keeps the oracle's
    expression order, so after K cycles p and every hist[k] equal the oracle's bit for bit (DESIGN.md §3 reading 12).
    The mean is summed in fp64 in a different order on the GPU; its fp32 rounding can differ only with probability ~1e-9
    (in fp64 the differently ordered sum itself shows in the last bits of p, so fp64 is held to 1e-10 only)."""
    torch, wl = env["torch"], env["wl"]
    cfg = env["synth"].make_config(config, dtype=dt, scale=scale)
    L, u = cfg["L"].astype(dt), cfg["u"].astype(dt)
    o = env["oracle"].Oracle(cfg["dims"], dt)
    o.set_coeff(L)
    b = o.divergence(u)
    p_ref, hist_ref, _, _ = o.solve(np.zeros_like(b), b, 0.0, K)
    pr = _projector(env, cfg, dt)
    wl.wl_set_coeff(pr.ctx, torch.from_numpy(L).cuda())
    bd = pr.empty_cells()
    wl.wl_divergence(pr.ctx, torch.from_numpy(u).cuda(), bd)
    assert bd.cpu().numpy().tobytes() == b.tobytes()
    p = pr.zeros_cells()
    hist, nc, rc = wl.wl_solve(pr.ctx, p, bd, 0.0, K)
    assert nc == K
    assert np.array_equal(hist, hist_ref), np.abs(hist / hist_ref - 1).max()
    assert p.cpu().numpy().tobytes() == p_ref.tobytes()
    pr.close()


@pytest.mark.parametrize("p", [4, 5])
def test_donut_grids_project_to_tolerance(env, p):
    """Paper-shaped 2:1:1 grids with a torus: full wl_project against the oracle — same
    cycle count, history and p bit-identical, corrected velocity within the fp32 bar, divergence reduced by 1e-4."""
    torch, wl = env["torch"], env["wl"]
    dt = np.float32
    cfg = env["synth"].make_donut(p)
    o = env["oracle"].Oracle(cfg["dims"], dt)
    shape = tuple(reversed(cfg["dims"]))
    u_ref, p_ref, hist_ref, nc_ref, rc_ref = o.project(cfg["u"], cfg["L"], np.zeros(shape, dt), cfg["tol"], cfg["maxcycles"])
    pr = _projector(env, cfg, dt)
    ud = torch.from_numpy(cfg["u"]).cuda()
    pd = pr.zeros_cells()
    hist, nc, rc = wl.wl_project(pr.ctx, ud, torch.from_numpy(cfg["L"]).cuda(), pd, cfg["tol"], cfg["maxcycles"])
    assert (nc, rc) == (nc_ref, rc_ref)
    assert np.array_equal(hist, hist_ref)
    assert pd.cpu().numpy().tobytes() == p_ref.tobytes()
    du = np.abs(ud.cpu().numpy() - u_ref).max() / np.abs(u_ref).max()
    assert du <= 1e-6
    if rc == 0:
        assert np.abs(o.divergence(ud.cpu().numpy())).max() <= 1.1e-4 * hist[0]
    pr.close()


@pytest.mark.parametrize("config,scale,far", [(2, 2, False), (2, 2, True), (1, 4, True), (3, 4, False)])
def test_warm_start_stop_reference_matches_oracle(env, config, scale, far):
    """The stop rule multiplies ||b||inf, not the initial residual (BJ "until ||r||inf <= 1e-4·||b||inf"; the oracle's
    reading is pinned by tests/test_oracle_cycle.py::test_stop_rule_reference_is_norm_of_b_not_initial_residual).  A warm
    start p0 != 0 separates the two norms: `far` = large noise (initial residual >> ||b||), otherwise a partially converged
    iterate with a constant offset (initial residual << ||b||).  Same cycle count, history and p as the oracle."""
    torch, wl = env["torch"], env["wl"]
    dt = np.float32
    cfg = env["synth"].make_config(config, dtype=dt, scale=scale)
    o = env["oracle"].Oracle(cfg["dims"], dt)
    o.set_coeff(cfg["L"])
    b = o.divergence(cfg["u"])
    shape = b.shape
    rng = np.random.default_rng(77 + config)
    if far:
        p0 = (50.0 * rng.standard_normal(shape)).astype(dt)
    else:
        p0, _, _, _ = o.solve(np.zeros(shape, dt), b, 0.0, 5)
        p0 = (p0 + dt(0.25)).astype(dt)
    _, r0 = o.residual(p0, b)
    nb = np.abs(b).max()
    assert (r0 > 20 * nb) if far else (r0 < 0.05 * nb)
    tol = 1e-3
    p_ref, hist_ref, nc_ref, rc_ref = o.solve(p0, b, tol, 32)
    assert hist_ref[0] == r0 and 0 < nc_ref
    pr = _projector(env, cfg, dt)
    wl.wl_set_coeff(pr.ctx, torch.from_numpy(cfg["L"]).cuda())
    bd = torch.from_numpy(b).cuda()
    p = torch.from_numpy(p0).cuda()
    hist, nc, rc = wl.wl_solve(pr.ctx, p, bd, tol, 32)
    assert (nc, rc) == (nc_ref, rc_ref), (nc, nc_ref, hist, hist_ref)
    _check_hist(hist, hist_ref, dt)
    _check_p(p.cpu().numpy(), p_ref, dt)
    if rc == 0:
        assert hist[-1] <= tol * nb < hist[-2]
    pr.close()
