"""Input generators: seeded, stateless, shaped as BASELINE.json `configs` say."""
import math

import numpy as np

from paper_2304_08159_b200 import synth


def test_mu0_values_and_shape():
    # BJ north_star: 0 for d <= -1, 1 for d >= 1, else 0.5 (1 + d + sin(pi d)/pi)
    assert synth.mu0(-1.0) == 0.0 and synth.mu0(-5.0) == 0.0
    assert synth.mu0(1.0) == 1.0 and synth.mu0(7.0) == 1.0
    assert synth.mu0(0.0) == 0.5
    assert abs(synth.mu0(0.5) - 0.5 * (1.5 + 1.0 / math.pi)) < 1e-15
    d = np.linspace(-1.5, 1.5, 3001)
    v = synth.mu0(d)
    assert v.min() >= 0.0 and v.max() <= 1.0
    assert np.all(np.diff(v) >= 0)                               # monotone
    assert np.abs(v + synth.mu0(-d) - 1.0).max() < 1e-15         # mu0(d) + mu0(-d) = 1
    # never negative just above d = -1 (c-8)
    assert synth.mu0(np.nextafter(-1.0, 0.0)) >= 0.0
    assert np.all(synth.mu0(-1.0 + np.logspace(-12, -4, 50)) >= 0.0)


def test_uniform_lattice_and_determinism():
    a = synth.uniform_pm1(123, 100000)
    b = synth.uniform_pm1(123, 100000)
    c = synth.uniform_pm1(124, 100000)
    assert a.dtype == np.float32 and np.array_equal(a, b) and not np.array_equal(a, c)
    assert np.all(np.abs(a) < 1.0) and np.all(a != 0.0)
    k = (a.astype(np.float64) + 1.0) * (1 << 24)
    assert np.all(k == np.round(k)) and np.all(k.astype(np.int64) % 2 == 1)  # odd lattice points, exact in fp32
    # stateless: any window equals the same slice of the full stream
    w = synth.uniform_pm1(123, 1000, start=5000)
    assert np.array_equal(w, a[5000:6000])
    assert abs(a.mean()) < 0.01 and abs(a.std() - 1 / math.sqrt(3)) < 0.01
    # chunking does not change values
    assert np.array_equal(synth.uniform_pm1(123, 100000, chunk=777), a)


def test_normal_moments():
    g = synth.normal(55, 200000, 1e-2)
    assert g.dtype == np.float64
    assert abs(g.mean()) < 1e-4 and abs(g.std() - 1e-2) < 1e-4
    assert np.array_equal(synth.normal(55, 100, 1e-2, start=1000), g[1000:1100])


def test_sphere_coeff_box_restricted_equals_brute_force():
    dims = (40, 36, 32)
    centres = [[12.0, 14.0, 15.5], [25.3, 20.1, 12.2], [30.0, 30.0, 28.0]]
    radii = [6.0, 7.5, 3.2]
    a = synth.coeff_spheres(dims, centres, radii, np.float32)
    b = synth.coeff_spheres(dims, centres, radii, np.float32, brute_force=True)
    assert np.array_equal(a, b)
    assert a.min() == 0.0 and a.max() == 1.0
    a2 = synth.coeff_spheres((48, 40), [[20.0, 18.0]], [9.0], np.float64)
    b2 = synth.coeff_spheres((48, 40), [[20.0, 18.0]], [9.0], np.float64, brute_force=True)
    assert np.array_equal(a2, b2)
    # face-centre convention: L[0] at (I0=20, I1=17) sits at x=(20, 17.5): distance 0.5 from the centre -> inside
    assert a2[0][17, 20] == 0.0
    # walls
    assert np.all(a2[0][:, 0] == 0) and np.all(a2[1][0, :] == 0)


def test_configs_shapes_and_masks():
    c0 = synth.make_config(0)
    assert c0["dims"] == (64, 64) and c0["L"].shape == (2, 64, 64) and c0["u"].dtype == np.float32
    assert c0["call"] == "solve" and c0["maxcycles"] == 10 and c0["tol"] == 0.0
    assert np.all(c0["u"][0][:, 0] == 0) and np.all(c0["u"][1][0, :] == 0)
    assert np.all(c0["L"][0][:, 1:] == 1)
    c1 = synth.make_config(1, scale=4)
    assert c1["dims"] == (256, 256)
    dead = (c1["L"][0] == 0).mean()
    assert 0.01 < dead < 0.08
    c2 = synth.make_config(2, scale=2)
    assert c2["dims"] == (64, 64, 64) and c2["call"] == "project"
    c3 = synth.make_config(3, scale=8)
    assert c3["dims"] == (32, 32, 32)
    # Taylor-Green at faces is discretely divergence-free: the divergence of u is all noise (c-17)
    u = c3["u"].astype(np.float64)
    assert 0.3 < np.abs(u[0]).max() < 1.1 and np.abs(u[2]).max() < 0.1
    c4 = synth.make_config(4, scale=8)
    assert c4["dims"] == (64, 64, 64)
    frac_partial = ((c4["L"] > 0) & (c4["L"] < 1)).mean()
    assert 0.0 < frac_partial < 0.2
    cen, rad = synth.sphere_params(4, (512, 512, 512))
    assert cen.shape == (32, 3) and rad.min() >= 8 and rad.max() <= 32
    assert cen.min() >= 32 and cen.max() <= 480


def test_donut_shape_and_coefficients():
    """Paper-shaped grid: 2:1:1 box, torus about the box centre; L = 0 deep inside the tube, 1 far away,
    symmetric under reflection of the transverse axes about the centre plane (cell-centred reflection)."""
    from paper_2304_08159_b200 import synth
    cfg = synth.make_donut(5)
    assert cfg["dims"] == (64, 32, 32) and cfg["L"].shape == (3, 32, 32, 64)
    L = cfg["L"].astype(np.float64)
    assert L.min() == 0.0 and L.max() == 1.0
    # a cell centre on the tube's centre circle: x = 32, y = 16 + 8, z = 16 -> faces around it are inside (r = 2)
    assert L[1, 16, 24, 32] == 0.0 and L[2, 16, 24, 32] == 0.0
    assert L[0, 2, 2, 5] == 1.0                                   # far corner: fluid
    assert np.all(L[0, :, :, 0] == 0) and np.all(L[1, :, 0, :] == 0) and np.all(L[2, 0, :, :] == 0)   # walls
    # component 0 (faces normal to the axis) is symmetric under z -> N2-1-z and y -> N1-1-y (cell-centred in y, z)
    assert np.array_equal(L[0], L[0][::-1, :, :]) and np.array_equal(L[0], L[0][:, ::-1, :])
    assert np.array_equal(cfg["u"], (synth.velocity_uniform(cfg["dims"], synth.seed_for(5, 5)) * cfg["L"]))
