"""T1/T2 — wl_set_bodies (device-side BDIM coefficients) against the oracle's body_coeff (pinned by
tests/test_oracle_body.py).  Bar (include/wl.h): identical except where device sin() and libm differ in the last bit of an
fp64 value — at most 1 ulp of fp32 (rarely: the cast hides it) / 4.5e-16 absolute in fp64, only on faces with |d| < 1; exact 0 / 1 and
exact wall planes everywhere else; the coarse levels are then the bit-exact sums of whatever level 0 holds."""
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


def _bodies_of(env, config, dims, scale):
    o, synth = env["oracle"], env["synth"]
    if config == 1:
        return o.body_records([(o.BODY_SPHERE, (256.0 / scale, 512.0 / scale), 64.0 / scale)])
    if config == 2:
        return o.body_records([(o.BODY_SPHERE, (48.0 / scale, 64.0 / scale, 64.0 / scale), 24.0 / scale)])
    if config == 4:
        c, r = synth.sphere_params(4, dims, scale=scale)
        return o.body_records([(o.BODY_SPHERE, ci, ri) for ci, ri in zip(c, r)])
    return np.zeros((0, 8))


def _check_level0(Lg, Lo, dt):
    assert Lg.shape == Lo.shape
    same = Lg == Lo
    frac = 1.0 - same.mean()
    if np.dtype(dt) == np.float32:
        assert frac <= 1e-4, frac                                   # last-bit sin() disagreements rarely survive the cast
    if not same.all():
        a, b = Lg[~same].astype(np.float64), Lo[~same].astype(np.float64)
        ulp = np.spacing(np.maximum(np.abs(a), np.abs(b)).astype(dt)).astype(np.float64)
        # the formula 0.5 (1 + d + sin(pi d)/pi) adds terms of size ~1: a last-bit difference of sin() (device <= 2 ulp, libm
        # <= 1 ulp) is an ABSOLUTE 1-2 ulp(1) of fp64 in the result, however small the result is (cancellation near d = -1)
        assert np.all(np.abs(a - b) <= np.maximum(ulp, 4.5e-16)) and np.all((b > 0) & (b < 1))
    assert np.all(Lg[Lo == 0.0] == 0.0) and np.all(Lg[Lo == 1.0] == 1.0)


@pytest.mark.parametrize("config,scale,dt", [(0, 1, np.float32), (1, 2, np.float32), (1, 4, np.float64), (2, 1, np.float32),
                                             (2, 2, np.float64), (4, 4, np.float32), (4, 8, np.float64)])
def test_level0_coefficients_and_hierarchy(env, config, scale, dt):
    torch, wl, o = env["torch"], env["wl"], env["oracle"]
    cfg = env["synth"].make_config(config, dtype=dt, scale=scale)
    dims = cfg["dims"]
    rec = _bodies_of(env, config, dims, scale)
    Lo = o.body_coeff(dims, dt, rec)
    assert np.array_equal(Lo, cfg["L"])                             # the oracle routine reproduces the config's input field
    pr = wl.Projector(dims, dt)
    wl.wl_set_bodies(pr.ctx, rec)
    Lg = pr.get_coeff(0).cpu().numpy()
    _check_level0(Lg, Lo, dt)
    # coarse levels: bit-exact sums of the GPU's own level 0 (the chain is wl_set_coeff's)
    orc = o.Oracle(dims, dt)
    orc.set_coeff(Lg)
    for l in range(pr.num_levels):
        assert pr.get_coeff(l).cpu().numpy().tobytes() == orc.get_coeff(l).tobytes(), l
    pr.close()


def test_torus_odd_shape_and_argument_checks(env):
    torch, wl, o = env["torch"], env["wl"], env["oracle"]
    cfg = env["synth"].make_donut(5)
    n1 = 32
    rec = o.body_records([(o.BODY_TORUS, (n1, n1 / 2, n1 / 2), n1 / 4.0, n1 / 16.0)])
    Lo = o.body_coeff(cfg["dims"], np.float32, rec)
    assert np.array_equal(Lo, cfg["L"])
    pr = wl.Projector(cfg["dims"], np.float32)
    wl.wl_set_bodies(pr.ctx, rec)
    _check_level0(pr.get_coeff(0).cpu().numpy(), Lo, np.float32)
    pr.close()
    # rows that are not whole 16-byte vectors take the any-shape kernel
    dims = (13, 10, 9)
    rec = o.body_records([(o.BODY_SPHERE, (6.2, 5.1, 4.4), 3.3), (o.BODY_TORUS, (7.0, 5.0, 4.5), 3.0, 1.0)])
    pr = wl.Projector(dims, np.float64)
    wl.wl_set_bodies(pr.ctx, rec)
    _check_level0(pr.get_coeff(0).cpu().numpy(), o.body_coeff(dims, np.float64, rec), np.float64)
    with pytest.raises(wl.WlError):
        wl.wl_set_bodies(pr.ctx, np.array([[7.0, 1, 1, 1, 1, 0, 0, 0]]))      # unknown kind
    with pytest.raises(wl.WlError):
        wl.wl_set_bodies(pr.ctx, np.array([[0.0, 1, 1, 1, -1.0, 0, 0, 0]]))   # negative radius
    pr.close()
    pr2 = wl.Projector((16, 16), np.float32)
    with pytest.raises(wl.WlError):
        wl.wl_set_bodies(pr2.ctx, np.array([[1.0, 8, 8, 0, 4, 1, 0, 0]]))     # torus in 2-D
    pr2.close()


def test_moving_body_projection_matches_the_oracle(env):
    """The use case: a body that moves between steps — wl_set_bodies + wl_project(L = NULL) per step, pressure warm-started.
    Each step is compared with the oracle fed the GPU's own level-0 coefficients (so the <= 1 ulp sin() differences of
    level 0 do not enter): same cycle counts, histories and fields within the fp32 bars."""
    torch, wl, o = env["torch"], env["wl"], env["oracle"]
    dt = np.float32
    dims = (64, 48, 32)
    rng = np.random.default_rng(11)
    u0 = rng.uniform(-1, 1, size=(3, 32, 48, 64)).astype(dt)
    pr = wl.Projector(dims, dt)
    orc = o.Oracle(dims, dt)
    p = pr.zeros_cells()
    p_ref = np.zeros(pr.cell_shape(), dt)
    for step in range(3):
        rec = o.body_records([(o.BODY_SPHERE, (20.0 + 2.5 * step, 24.0, 16.0 + 0.5 * step), 7.0)])
        wl.wl_set_bodies(pr.ctx, rec)
        Lg = pr.get_coeff(0).cpu().numpy()
        _check_level0(Lg, o.body_coeff(dims, dt, rec), dt)
        u = (u0 * Lg).astype(dt)
        ud = torch.from_numpy(u).cuda()
        hist, nc, rc = wl.wl_project(pr.ctx, ud, None, p, 1e-4, 32)
        u_ref, p_ref, hist_ref, nc_ref, rc_ref = orc.project(u, Lg, p_ref, 1e-4, 32)
        assert (nc, rc) == (nc_ref, rc_ref)
        assert np.abs(hist / hist_ref - 1.0).max() <= 1e-3
        assert np.abs(p.cpu().numpy() - p_ref).max() <= 1e-4 * np.abs(p_ref).max()
        assert np.abs(ud.cpu().numpy() - u_ref).max() <= 1e-4 * np.abs(u_ref).max()
    pr.close()


def test_config4_full_512_thirty_two_spheres(env):
    """wl_set_bodies at the size and body count bench.py's `e2e` leg runs it on every step (BASELINE configs[4]: 512^3 fp32, 32
    seeded spheres; Table 2 `BDIM!`): level 0 against oracle.body_coeff face by face, every coarse level
    bit-exact against the oracle's coarsening of the GPU's own level 0."""
    torch, wl, o = env["torch"], env["wl"], env["oracle"]
    dt = np.float32
    cfg = env["synth"].make_config(4, dtype=dt)
    dims = cfg["dims"]
    rec = _bodies_of(env, 4, dims, 1)
    assert rec.shape == (32, 8) and int(np.prod(dims)) == 512 ** 3
    Lo = o.body_coeff(dims, dt, rec)
    assert np.array_equal(Lo, cfg["L"])
    pr = wl.Projector(dims, dt)
    wl.wl_set_bodies(pr.ctx, rec)
    Lg = pr.get_coeff(0).cpu().numpy()
    _check_level0(Lg, Lo, dt)
    del Lo
    orc = o.Oracle(dims, dt)
    orc.set_coeff(Lg)
    for l in range(pr.num_levels):
        assert pr.get_coeff(l).cpu().numpy().tobytes() == orc.get_coeff(l).tobytes(), l
    pr.close()
