"""T0 pins for coefficient coarsening, restriction and prolongation (BJ north_star: "Restriction R sums the 2^n
children; prolongation P is piecewise-constant injection"; "A_c = R·A·P exactly")."""
import numpy as np
import pytest

from dense_ref import dense_from_apply, incidence_laplacian, random_coeff, restriction_matrix

GRIDS = [(8, 8), (8, 16), (16, 8), (8, 8, 8), (16, 8, 8), (8, 8, 16)]


def _dense_ops(o, level):
    fs, cs = o.cell_shape(level), o.cell_shape(level + 1)
    M, Mc = int(np.prod(fs)), int(np.prod(cs))
    R = np.zeros((Mc, M))
    e = np.zeros(M)
    for j in range(M):
        e[j] = 1
        R[:, j] = o.restrict(e.reshape(fs), level).ravel()
        e[j] = 0
    P = np.zeros((M, Mc))
    e = np.zeros(Mc)
    for j in range(Mc):
        e[j] = 1
        P[:, j] = o.prolong_add(e.reshape(cs), np.zeros(fs), level).ravel()
        e[j] = 0
    return R, P


@pytest.mark.parametrize("dims", GRIDS)
def test_R_is_child_sum_P_is_injection_and_galerkin(oracle_mod, dims):
    rng = np.random.default_rng(21 + dims[0] + 7 * len(dims))
    L = random_coeff(dims, rng)
    o = oracle_mod.Oracle(dims, np.float64)
    o.set_coeff(L)
    assert o.num_levels >= 2
    R, P = _dense_ops(o, 0)
    assert np.array_equal(R, restriction_matrix(dims))
    assert np.array_equal(R, P.T)                    # R = P^T exactly
    assert np.array_equal(P.sum(axis=1), np.ones(P.shape[0]))  # each fine cell has one parent
    A = incidence_laplacian(dims, L)
    cd = o.level_dims(1)
    Ac_galerkin = R @ A @ P
    # (i) the oracle's coarse operator applied cell by cell
    cs = o.cell_shape(1)
    Ac_oracle = dense_from_apply(lambda e: o.apply_A(e.reshape(cs), 1).ravel(), int(np.prod(cs)))
    assert np.abs(Ac_oracle - Ac_galerkin).max() <= 2e-14
    # (ii) the coarsened coefficients themselves, through the independent incidence form
    Lc = o.get_coeff(1)
    assert np.abs(incidence_laplacian(cd, Lc) - Ac_galerkin).max() <= 2e-14


@pytest.mark.parametrize("dims", [(16, 16), (16, 16, 16), (32, 16, 8)])
def test_uniform_L_coarsens_to_powers_of_two(oracle_mod, dims):
    from paper_2304_08159_b200 import synth
    n = len(dims)
    for dt in (np.float32, np.float64):
        o = oracle_mod.Oracle(dims, dt)
        o.set_coeff(synth.coeff_uniform(dims, dt))
        for lev in range(o.num_levels):
            Lc = o.get_coeff(lev)
            expect = synth.coeff_uniform(o.level_dims(lev), dt) * dt(2.0 ** ((n - 1) * lev))
            assert np.array_equal(Lc, expect)


@pytest.mark.parametrize("dims", [(16, 8), (8, 16, 8)])
def test_dyadic_L_coarsening_is_exact_in_any_order(oracle_mod, dims):
    """Multiples of 2^-10 sum exactly in fp32, so the result is order-independent: catches indexing errors."""
    rng = np.random.default_rng(33)
    n = len(dims)
    L = random_coeff(dims, rng, dtype=np.float32, dyadic=True)
    o = oracle_mod.Oracle(dims, np.float32)
    o.set_coeff(L)
    Lc = o.get_coeff(1)
    L64 = L.astype(np.float64)
    for i in range(n):
        # sum over the children with c_i = 0: take even index along axis i, sum pairs along the others
        ref = L64[i]
        for a in range(n):
            ax = n - 1 - a
            if a == i:
                ref = np.take(ref, np.arange(0, dims[a], 2), axis=ax)
            else:
                sh = list(ref.shape)
                sh[ax] = dims[a] // 2
                sh.insert(ax + 1, 2)
                ref = ref.reshape(sh).sum(axis=ax + 1)
        assert np.array_equal(Lc[i].astype(np.float64), ref)


def test_level_table_rule(oracle_mod):
    """Coarsen while every extent is even and every half >= 4 (c-3, c-4); BASELINE configs' level counts."""
    cases = {(64, 64): 5, (1024, 1024): 9, (128, 128, 128): 6, (8, 4, 4): 1, (12, 8): 2, (32, 16, 16): 3,
             (5, 7): 1, (24, 24): 3}
    for dims, grids in cases.items():
        o = oracle_mod.Oracle(dims, np.float32)
        assert o.num_levels == grids, dims
        last = o.level_dims(grids - 1)
        assert all(d >= 4 for d in last)
    o = oracle_mod.Oracle((64, 64), np.float32)
    assert o.level_dims(4) == (4, 4)
    with pytest.raises(ValueError):
        oracle_mod.Oracle((3, 8), np.float32)


def test_divergence_and_gradient_are_incidence_transposes(oracle_mod):
    """H1: b = D u with D = -G^T on interior faces (+ wall faces contributing u at I_i = 0);
    H8: u -= L * (G p) on interior faces, wall plane untouched."""
    dims = (6, 5, 4)
    n = 3
    rng = np.random.default_rng(4)
    shape = tuple(reversed(dims))
    u = rng.standard_normal((n,) + shape)
    p = rng.standard_normal(shape)
    L = random_coeff(dims, rng)
    o = oracle_mod.Oracle(dims, np.float64)
    o.set_coeff(L)
    b = o.divergence(u)
    ref = np.zeros(shape)
    for i in range(n):
        ax = n - 1 - i
        up = np.zeros(shape)
        dst = [slice(None)] * n
        src = [slice(None)] * n
        dst[ax] = slice(0, dims[i] - 1)
        src[ax] = slice(1, dims[i])
        up[tuple(dst)] = u[i][tuple(src)]
        ref += up - u[i]
    assert np.abs(b - ref).max() <= 1e-14
    u2 = o.gradient_correct(u, p)
    for i in range(n):
        ax = n - 1 - i
        g = np.zeros(shape)
        dst = [slice(None)] * n
        src = [slice(None)] * n
        dst[ax] = slice(1, dims[i])
        src[ax] = slice(0, dims[i] - 1)
        g[tuple(dst)] = p[tuple(dst)] - p[tuple(src)]
        assert np.abs(u2[i] - (u[i] - L[i] * g)).max() <= 1e-14
        wall = [slice(None)] * n
        wall[ax] = 0
        assert np.array_equal(u2[i][tuple(wall)], u[i][tuple(wall)])
    # div(u - L grad p) = div u - A p   (the identity the projection rests on)
    A = incidence_laplacian(dims, L)
    # wall planes of u are not masked here, so compare differences: div(u) - div(u2) = A p
    assert np.abs((b - o.divergence(u2)).ravel() - A @ p.ravel()).max() <= 1e-13
