"""T0 pins for the oracle's operator A, diagonal and Jacobi sweep (SURVEY.md §8(c) "What pins the oracle").

Every expected value below is built WITHOUT the oracle: a Kronecker-sum textbook Neumann Laplacian, a
face-incidence form -G^T diag(L) G, closed-form cosine eigenpairs, dense NumPy algebra.
"""
import math

import numpy as np
import pytest

from dense_ref import dense_from_apply, incidence_laplacian, random_coeff

GRIDS = [(8, 8), (8, 4), (12, 8), (5, 7), (8, 8, 8), (8, 4, 4), (6, 5, 4)]


def _oracle(oracle_mod, dims, L, dtype=np.float64):
    o = oracle_mod.Oracle(dims, dtype)
    o.set_coeff(L)
    return o


def _dense_A(o):
    M = int(np.prod(o.dims))
    shape = o.cell_shape(0)
    return dense_from_apply(lambda e: o.apply_A(e.reshape(shape)).ravel(), M)


def neumann_1d(N):
    """Textbook 1-D Neumann (zero-flux walls) second-difference matrix: rows sum to zero."""
    T = np.zeros((N, N))
    for k in range(N):
        if k > 0:
            T[k, k - 1] = 1.0
            T[k, k] -= 1.0
        if k < N - 1:
            T[k, k + 1] = 1.0
            T[k, k] -= 1.0
    return T


@pytest.mark.parametrize("dims", GRIDS)
def test_uniform_L_is_kronecker_sum_neumann_laplacian(oracle_mod, dims):
    from paper_2304_08159_b200 import synth
    o = _oracle(oracle_mod, dims, synth.coeff_uniform(dims, np.float64))
    A = _dense_A(o)
    n = len(dims)
    # linear index = I_0 + N_0 (I_1 + N_1 I_2): axis 0 is the fastest => last Kronecker factor
    ref = np.zeros_like(A)
    for i in range(n):
        mats = [np.eye(dims[j]) for j in range(n)]
        mats[i] = neumann_1d(dims[i])
        K = np.array([[1.0]])
        for j in reversed(range(n)):  # slowest axis first
            K = np.kron(K, mats[j])
        ref += K
    assert np.array_equal(A, ref)


@pytest.mark.parametrize("dims", GRIDS)
def test_variable_L_matches_incidence_form_and_structure(oracle_mod, dims):
    rng = np.random.default_rng(7 + len(dims) * 100 + dims[0])
    L = random_coeff(dims, rng)
    o = _oracle(oracle_mod, dims, L)
    A = _dense_A(o)
    ref = incidence_laplacian(dims, L)
    assert np.abs(A - ref).max() <= 4e-15
    # symmetry, A·1 = 0, negative semi-definite, diag = -D
    assert np.abs(A - A.T).max() <= 1e-15
    assert np.abs(A @ np.ones(A.shape[0])).max() <= 4e-15
    assert np.linalg.eigvalsh(0.5 * (A + A.T)).max() <= 1e-13
    n = len(dims)
    D = np.zeros(tuple(reversed(dims)))
    for i in range(n):
        ax = n - 1 - i
        D += L[i]  # lower face (wall plane already 0)
        up = np.zeros_like(D)
        sl_dst = [slice(None)] * n
        sl_src = [slice(None)] * n
        sl_dst[ax] = slice(0, dims[i] - 1)
        sl_src[ax] = slice(1, dims[i])
        up[tuple(sl_dst)] = L[i][tuple(sl_src)]
        D += up
    assert np.abs(np.diag(A) + D.ravel()).max() <= 4e-15


def test_wall_plane_of_caller_L_is_ignored(oracle_mod):
    """set_coeff forces the stored wall plane I_i = 0 to zero in its own copy (c-6)."""
    dims = (8, 6)
    rng = np.random.default_rng(3)
    L = random_coeff(dims, rng)
    Ldirty = L.copy()
    Ldirty[0][:, 0] = 0.7
    Ldirty[1][0, :] = 0.3
    a = _dense_A(_oracle(oracle_mod, dims, L))
    b = _dense_A(_oracle(oracle_mod, dims, Ldirty))
    assert np.array_equal(a, b)
    assert np.array_equal(_oracle(oracle_mod, dims, Ldirty).get_coeff(0), L)


@pytest.mark.parametrize("dims,k", [((16, 16), (1, 2)), ((8, 12), (3, 0)), ((8, 8, 8), (1, 2, 3)), ((16, 8, 4), (2, 1, 0))])
def test_cosine_modes_are_eigenvectors_closed_form(oracle_mod, dims, k):
    """p = prod cos(pi k_i x_i / N_i), x_i = I_i + 1/2, uniform L: A p = lambda p, lambda = sum 2cos(pi k_i/N_i) - 2 (c-24)."""
    from paper_2304_08159_b200 import synth
    n = len(dims)
    o = _oracle(oracle_mod, dims, synth.coeff_uniform(dims, np.float64))
    p = np.ones(tuple(reversed(dims)))
    lam = 0.0
    for i in range(n):
        x = np.arange(dims[i]) + 0.5
        c = np.cos(math.pi * k[i] * x / dims[i])
        shape = [1] * n
        shape[n - 1 - i] = dims[i]
        p = p * c.reshape(shape)
        lam += 2.0 * math.cos(math.pi * k[i] / dims[i]) - 2.0
    Ap = o.apply_A(p)
    assert np.abs(Ap - lam * p).max() <= 2e-15 * max(1.0, abs(lam)) * 4
    if (dims, k) == ((16, 16), (1, 2)):
        assert abs(lam - (-0.190670)) < 1e-6  # value quoted in SURVEY.md Appendix A.1


@pytest.mark.parametrize("dims", [(8, 8), (12, 8), (8, 4, 4)])
def test_jacobi_sweep_matches_dense_formula(oracle_mod, dims):
    """x' = x + w D^-1 (A x - b), w = 2/3, all cells from the old x; cells with D = 0 are left unchanged."""
    rng = np.random.default_rng(11)
    L = random_coeff(dims, rng)
    # make one cell dead (all its faces zero) to exercise invD = 0
    n = len(dims)
    dead = tuple(2 for _ in range(n))  # NumPy index
    for i in range(n):
        L[(i,) + dead] = 0.0
        up = list(dead)
        up[n - 1 - i] += 1
        L[(i,) + tuple(up)] = 0.0
    o = _oracle(oracle_mod, dims, L)
    A = incidence_laplacian(dims, L)
    D = -np.diag(A)
    assert D[np.ravel_multi_index(dead, tuple(reversed(dims)))] == 0.0
    invD = np.where(D > 0, 1.0 / np.where(D > 0, D, 1.0), 0.0)
    x = rng.standard_normal(A.shape[0])
    b = rng.standard_normal(A.shape[0])
    shape = tuple(reversed(dims))
    ref = x.copy()
    for s in range(1, 4):
        ref = ref + (2.0 / 3.0) * invD * (A @ ref - b)
        got = o.jacobi(x.reshape(shape), b.reshape(shape), s).ravel()
        assert np.abs(got - ref).max() <= 1e-14 * max(1.0, np.abs(ref).max())
    # Jacobi is not Gauss-Seidel: a sweep must not see its own updates (checked by the dense formula above
    # and by symmetry of the response to a centred impulse on a uniform grid)


def test_residual_and_norm(oracle_mod):
    dims = (8, 6, 4)
    rng = np.random.default_rng(5)
    L = random_coeff(dims, rng)
    o = _oracle(oracle_mod, dims, L)
    A = incidence_laplacian(dims, L)
    x = rng.standard_normal(A.shape[0])
    b = rng.standard_normal(A.shape[0])
    shape = tuple(reversed(dims))
    r, nrm = o.residual(x.reshape(shape), b.reshape(shape))
    ref = b - A @ x
    assert np.abs(r.ravel() - ref).max() <= 1e-14
    assert nrm == np.abs(r).max()


def test_fp32_operator_close_to_fp64(oracle_mod):
    dims = (8, 8, 8)
    rng = np.random.default_rng(9)
    L = random_coeff(dims, rng).astype(np.float32)
    x = rng.standard_normal(tuple(reversed(dims))).astype(np.float32)
    y32 = _oracle(oracle_mod, dims, L, np.float32).apply_A(x)
    y64 = _oracle(oracle_mod, dims, L.astype(np.float64), np.float64).apply_A(x.astype(np.float64))
    assert y32.dtype == np.float32
    assert np.abs(y32 - y64).max() <= 2e-6
