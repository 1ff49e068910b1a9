"""T0 pins for the oracle's BDIM coefficient routine: L = mu0(signed distance at the face centre),
BASELINE.json north_star "BDIM face coefficient", SURVEY §8(c) c-8 / c-9.  Pinned by what the formula and the geometry fix:
special values and symmetry of mu0, exact 0 / 1 away from the interface, the face-centre convention on faces whose distance
is known in closed form, the lattice sum of 1 - L against the volume of the body, the min rule for several bodies."""
import math

import numpy as np
import pytest


def test_mu0_special_values_symmetry_monotonicity(oracle_mod):
    mu0 = oracle_mod.mu0
    assert mu0(-1.0) == 0.0 and mu0(1.0) == 1.0 and mu0(0.0) == 0.5
    assert mu0(-7.0) == 0.0 and mu0(3.0) == 1.0 and mu0(-1.0 - 1e-12) == 0.0 and mu0(1.0 + 1e-12) == 1.0
    assert abs(mu0(0.5) - (0.75 + 0.5 / math.pi)) <= 1e-15          # sin(pi/2) = 1
    assert abs(mu0(-0.5) - (0.25 - 0.5 / math.pi)) <= 1e-15
    ds = np.linspace(-1.0, 1.0, 2001)
    v = np.array([mu0(d) for d in ds])
    assert np.all(np.diff(v) >= 0) and v.min() >= 0.0 and v.max() <= 1.0
    assert np.abs(v + v[::-1] - 1.0).max() <= 1e-15                   # mu0(d) + mu0(-d) = 1
    assert mu0(-1.0 + 1e-4) <= 1e-11 and 1.0 - mu0(1.0 - 1e-4) <= 1e-11   # C^1 (in fact C^2) contact with 0 and 1
    # never negative just inside d = -1, where the formula cancels catastrophically (SURVEY c-8)
    assert min(mu0(-1.0 + k * 1e-7) for k in range(1, 200)) >= 0.0


def test_exact_zero_and_one_away_from_the_interface_and_zero_walls(oracle_mod):
    dims, c, R = (24, 20, 16), (11.3, 9.7, 8.1), 5.4
    L = oracle_mod.body_coeff(dims, np.float32, oracle_mod.body_records([(oracle_mod.BODY_SPHERE, c, R)]))
    assert L.shape == (3, 16, 20, 24) and L.min() >= 0.0 and L.max() <= 1.0
    for i in range(3):
        ax = [np.arange(dims[j], dtype=np.float64) + (0.0 if j == i else 0.5) for j in range(3)]
        X, Y, Z = np.meshgrid(ax[0], ax[1], ax[2], indexing="ij")        # (x, y, z) order
        dist = np.sqrt((X - c[0]) ** 2 + (Y - c[1]) ** 2 + (Z - c[2]) ** 2).transpose(2, 1, 0)
        Li = L[i].copy()
        wall = [slice(None)] * 3
        wall[2 - i] = 0
        assert np.all(Li[tuple(wall)] == 0.0)                            # stored wall plane I_i = 0
        inner = [slice(None)] * 3
        inner[2 - i] = slice(1, None)
        Li, di = Li[tuple(inner)], dist[tuple(inner)]
        assert np.all(Li[di >= R + 1.0] == 1.0) and np.all(Li[di <= R - 1.0] == 0.0)
        band = (di > R - 1.0) & (di < R + 1.0)
        assert band.any() and np.all(Li[band] >= 0.0) and np.all(Li[band] <= 1.0)
        assert np.all(np.diff(Li[band][np.argsort(di[band])]) >= -1e-7)   # monotone in the distance


def test_face_centre_convention(oracle_mod):
    """A small sphere centred exactly ON the centre of face ((8,8,8), i=0) = point (8, 8.5, 8.5): the distances of the
    neighbouring face centres are known in closed form."""
    dims, R = (16, 16, 16), 0.5
    L = oracle_mod.body_coeff(dims, np.float64, oracle_mod.body_records([(0, (8.0, 8.5, 8.5), R)]))
    f = lambda d: 0.5 * (1.0 + d + math.sin(math.pi * d) / math.pi)
    assert abs(L[0, 8, 8, 8] - f(0.0 - R)) <= 1e-15                  # the face the centre sits on: distance 0
    assert abs(L[0, 8, 8, 9] - f(1.0 - R)) <= 1e-15 and abs(L[0, 8, 8, 7] - f(1.0 - R)) <= 1e-15   # one cell along x
    assert L[0, 8, 9, 8] == f(1.0 - R) or abs(L[0, 8, 9, 8] - f(1.0 - R)) <= 1e-15                  # one cell along y
    d1 = math.sqrt(0.5 * 0.5 + 0.5 * 0.5) - R                        # faces of direction 1 around it: (8.5, 8 or 9, 8.5)
    for (z, y, x) in [(8, 8, 8), (8, 9, 8), (8, 8, 7), (8, 9, 7)]:
        assert abs(L[1, z, y, x] - f(d1)) <= 1e-15
    for (z, y, x) in [(8, 8, 8), (9, 8, 8), (8, 8, 7), (9, 8, 7)]:   # direction 2: (8.5, 8.5, 8 or 9)
        assert abs(L[2, z, y, x] - f(d1)) <= 1e-15
    # 2-D: a circle on the centre of face ((6,5), i=1) = point (6.5, 5)
    L2 = oracle_mod.body_coeff((12, 12), np.float64, oracle_mod.body_records([(0, (6.5, 5.0), R)]))
    assert abs(L2[1, 5, 6] - f(-R)) <= 1e-15 and abs(L2[1, 6, 6] - f(1.0 - R)) <= 1e-15 and abs(L2[0, 5, 6] - f(d1)) <= 1e-15


@pytest.mark.parametrize("R", [6.0, 9.5])
def test_lattice_sum_reproduces_the_volume(oracle_mod, R):
    """1 - mu0 is the body indicator smeared over +-1 cell with the kernel mu0'(d) = (1 + cos(pi d))/2, whose second moment
    is 1/3 - 2/pi^2: the integral of 1 - mu0(|x| - R) over space is 4/3 pi R^3 + 4 pi R (1/3 - 2/pi^2) exactly, and the
    lattice sum over any face family reproduces it (a flipped sign or a wrong smearing width moves it by O(R^2))."""
    dims, c = (40, 36, 32), (19.3, 18.1, 16.4)
    L = oracle_mod.body_coeff(dims, np.float64, oracle_mod.body_records([(0, c, R)]))
    vol = 4.0 / 3.0 * math.pi * R ** 3 + 4.0 * math.pi * R * (1.0 / 3.0 - 2.0 / math.pi ** 2)
    for i in range(3):
        inner = [slice(None)] * 3
        inner[2 - i] = slice(1, None)
        s = (1.0 - L[i][tuple(inner)]).sum()
        assert abs(s / vol - 1.0) <= 2e-3, (i, s, vol)
    # the centre of mass of 1 - L sits at the sphere's centre (each face family with its own half-cell offsets)
    for i in range(3):
        w = 1.0 - L[i]
        w[(slice(None),) * (2 - i) + (0,)] = 0.0
        for j in range(3):
            coord = np.arange(dims[j], dtype=np.float64) + (0.0 if j == i else 0.5)
            sh = [1, 1, 1]
            sh[2 - j] = dims[j]
            com = (w * coord.reshape(sh)).sum() / w.sum()
            assert abs(com - c[j]) <= 0.02, (i, j, com)


def test_several_bodies_take_the_minimum_distance_and_torus_surface(oracle_mod):
    dims = (32, 24, 24)
    a = (oracle_mod.BODY_SPHERE, (10.2, 11.0, 12.5), 4.3)
    b = (oracle_mod.BODY_SPHERE, (15.0, 13.0, 11.0), 3.1)           # overlaps a
    t = (oracle_mod.BODY_TORUS, (16.0, 8.5, 8.5), 4.0, 1.0)
    La = oracle_mod.body_coeff(dims, np.float64, oracle_mod.body_records([a]))
    Lb = oracle_mod.body_coeff(dims, np.float64, oracle_mod.body_records([b]))
    Lt = oracle_mod.body_coeff(dims, np.float64, oracle_mod.body_records([t]))
    Lall = oracle_mod.body_coeff(dims, np.float64, oracle_mod.body_records([a, b, t]))
    assert np.array_equal(Lall, np.minimum(np.minimum(La, Lb), Lt))    # mu0 is monotone: mu0(min d) = min mu0(d)
    L0 = oracle_mod.body_coeff(dims, np.float32, np.zeros((0, 8)))
    assert L0[0][:, :, 1:].min() == 1.0 and L0[0][:, :, 0].max() == 0.0  # no body: the uniform coefficient field
    # torus about axis 0, ring of radius 4 in the (1,2) plane, tube radius 1: face ((16, 13, 8), i=0) has its centre
    # (16, 13.5, 8.5) exactly on the tube surface (d = 0), ((16, 12, 8), 0) on the centre line (d = -1)
    assert abs(Lt[0, 8, 13, 16] - 0.5) <= 1e-15 and Lt[0, 8, 12, 16] == 0.0
    assert abs(Lt[0, 8, 14, 16] - 1.0) <= 1e-15                          # one cell further out: d = 1
