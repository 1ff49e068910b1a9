"""The pieces composed the way the paper's time step uses them (`convdiff!`, `BDIM!`, `project!` per step): a few
forward-Euler momentum steps  u* = u + dt convdiff(u);  u* <- L o u*  (the harness's BDIM masking, reading 9);
wl_project(u*, p) warm-started from the previous pressure, with the body's coefficients evaluated on the device (wl_set_bodies).
Every operation between the library calls is a single IEEE multiply or add on both sides, so the GPU sequence must reproduce
the oracle's: velocities and pressures after three steps bit for bit (fp32), cycle counts equal."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def test_three_momentum_steps_match_the_oracle(oracle_mod):
    import torch
    from paper_2304_08159_b200 import binding as wl, build, synth
    build.build_cuda()
    cfg = synth.make_config(2, scale=2)          # 64^3, one sphere
    dims, dt_ = cfg["dims"], np.float32
    nu, dt = 0.01, np.float32(0.05)
    pr = wl.Projector(dims, dt_)
    wl.wl_set_bodies(pr.ctx, cfg["bodies"])
    Ld = pr.get_coeff(0)                          # the coefficients the device built (level 0)
    L = Ld.cpu().numpy()
    o = oracle_mod.Oracle(dims, dt_)
    o.set_coeff(L)
    u_ref = cfg["u"].astype(dt_).copy()
    p_ref = np.zeros(tuple(reversed(dims)), dt_)
    u = torch.from_numpy(u_ref).cuda()
    p = pr.zeros_cells()
    r = torch.empty_like(u)
    for step in range(3):
        # oracle
        rr = oracle_mod.convdiff(u_ref, nu)
        us = (u_ref + dt * rr).astype(dt_)
        us = (L * us).astype(dt_)
        u_ref, p_ref, hist_ref, nc_ref, rc_ref = o.project(us, None, p_ref, 1e-4, 32)
        # GPU
        wl.wl_convdiff(pr.ctx, u, nu, r)
        us_d = u + r * float(dt)                  # two separately rounded elementwise kernels (no fused multiply-add)
        us_d = Ld * us_d
        hist, nc, rc = wl.wl_project(pr.ctx, us_d, None, p, 1e-4, 32)
        u = us_d
        assert (nc, rc) == (nc_ref, rc_ref), (step, nc, nc_ref)
        assert np.array_equal(hist, hist_ref), step
        assert np.array_equal(u.cpu().numpy(), u_ref), step
        assert p.cpu().numpy().tobytes() == p_ref.tobytes(), step
    assert np.isfinite(u_ref).all() and np.abs(u_ref).max() < 10.0
    pr.close()
