"""T0 pins for the oracle's V-cycle-preconditioned conjugate-gradient solve (PAPER.md:38
"Conjugate-Gradient smoothing within the GMG levels"; DESIGN.md §3 reading 13).

Nothing here retypes the oracle's loop: the reference is textbook preconditioned CG (Hestenes–Stiefel with a fixed SPD
preconditioner) written with DENSE NumPy matrices — the operator from the incidence form of tests/dense_ref.py, the
preconditioner = the dense-matrix multigrid recursion of tests/test_oracle_cycle.py applied to unit vectors — plus what
the mathematics of CG fixes: M^-1-orthogonal residuals, A-conjugate directions, monotone energy error, termination on
the pseudo-inverse solution in at most rank(A) steps.
"""
import numpy as np
import pytest

from dense_ref import incidence_laplacian, random_coeff
from test_oracle_cycle import dense_hierarchy, dense_vcycle


def dense_preconditioner(As, Rs):
    """The V-cycle from a zero guess is a linear map r -> z; its matrix, column by column."""
    M = As[0].shape[0]
    V = np.zeros((M, M))
    e = np.zeros(M)
    for j in range(M):
        e[j] = 1.0
        V[:, j] = dense_vcycle(As, Rs, 0, np.zeros(M), e)
        e[j] = 0.0
    return V


def dense_pcg(A, V, x0, b, iters):
    """Textbook PCG on A x = b (A symmetric negative semi-definite: the two sign changes of CG on -A cancel), with
    the mean of every preconditioned residual removed.  Returns the iterates, residuals, z's and directions."""
    x, r = x0.copy(), b - A @ x0
    xs, rs, zs, ps = [x.copy()], [r.copy()], [], []
    p, rho = None, None
    for k in range(iters):
        z = V @ r
        rho_new = r @ z
        z = z - z.mean()
        p = z if p is None else z + (rho_new / rho) * p
        rho = rho_new
        q = A @ p
        alpha = rho / (p @ q)
        x = x + alpha * p
        r = r - alpha * q
        xs.append(x.copy()); rs.append(r.copy()); zs.append(z.copy()); ps.append(p.copy())
    return xs, rs, zs, ps


def _case(oracle_mod, dims, seed, body=False):
    from paper_2304_08159_b200 import synth
    rng = np.random.default_rng(seed)
    n = len(dims)
    shape = tuple(reversed(dims))
    L = synth.coeff_spheres(dims, [[d / 2.0 for d in dims]], [min(dims) / 4.0], np.float64) if body else random_coeff(dims, rng)
    As, Rs = dense_hierarchy(dims, L)
    o = oracle_mod.Oracle(dims, np.float64)
    o.set_coeff(L)
    u = rng.standard_normal((n,) + shape) * L
    b = o.divergence(u).ravel()
    return o, As, Rs, b, shape, rng


@pytest.mark.parametrize("dims,body", [((8, 8), False), ((16, 8), False), ((8, 8, 8), False), ((8, 4, 4), False), ((16, 16), True)])
def test_pcg_iterates_equal_dense_textbook_pcg(oracle_mod, dims, body):
    o, As, Rs, b, shape, rng = _case(oracle_mod, dims, 400 + dims[0] + len(dims), body)
    A = As[0]
    V = dense_preconditioner(As, Rs)
    assert np.abs(V - V.T).max() <= 1e-12 * np.abs(V).max()          # the cycle is a symmetric preconditioner ...
    live = -np.diag(A) > 0
    Vl = V[np.ix_(live, live)]
    assert np.linalg.eigvalsh(0.5 * (Vl + Vl.T)).max() < 0           # ... and definite (like A^-1) on the live cells
    x0 = rng.standard_normal(b.size)
    K = 6
    xs, rs, zs, ps = dense_pcg(A, V, x0, b, K)
    for k in range(0, K + 1):
        p, hist, nit, rc = o.solve_pcg(x0.reshape(shape), b.reshape(shape), 0.0, k)
        assert nit == k and hist.shape == (k + 1,)
        ref = xs[k] - xs[k].mean()
        assert np.abs(p.ravel() - ref).max() <= 1e-10 * max(1.0, np.abs(ref).max()), k
        for j in range(k + 1):
            assert abs(hist[j] - np.abs(rs[j]).max()) <= 1e-10 * np.abs(rs[0]).max(), (k, j)
    # what CG itself guarantees of the reference the oracle has just been matched against
    for i in range(K):
        for j in range(i):
            assert abs(rs[i] @ (V @ rs[j])) <= 1e-8 * abs(rs[j] @ (V @ rs[j]))      # M^-1-orthogonal residuals
            assert abs(ps[i] @ (A @ ps[j])) <= 1e-8 * abs(ps[j] @ (A @ ps[j]))      # A-conjugate directions


@pytest.mark.parametrize("dims", [(4, 4), (8, 4), (4, 4, 4)])
def test_pcg_terminates_on_the_pseudo_inverse_solution(oracle_mod, dims):
    """CG minimises the energy error over a Krylov space that grows by one dimension per step: on M cells (rank M-1) it
    has the exact solution after at most M-1 steps; the energy error decreases monotonically on the way."""
    o, As, Rs, b, shape, rng = _case(oracle_mod, dims, 500 + dims[0] + len(dims))
    A = As[0]
    M = b.size
    xstar = np.linalg.pinv(A) @ b
    xstar -= xstar.mean()
    p, hist, nit, rc = o.solve_pcg(np.zeros(shape), b.reshape(shape), 1e-12, M)
    assert rc == 0 and nit <= M - 1
    assert np.abs(p.ravel() - xstar).max() <= 1e-9 * np.abs(xstar).max()
    assert abs(p.mean()) <= 1e-14
    prev = None
    for k in range(0, min(nit, 8) + 1):
        pk, _, _, _ = o.solve_pcg(np.zeros(shape), b.reshape(shape), 0.0, k)
        e = pk.ravel() - xstar
        en = -(e @ (A @ e))
        assert en >= -1e-14
        if prev is not None:
            assert en <= prev * (1 + 1e-12)
        prev = en


def test_pcg_needs_fewer_applications_of_the_cycle_than_plain_cycling(oracle_mod):
    """Same answer as SOLVE (the dense pseudo-inverse solution on live cells), in fewer V-cycles."""
    from paper_2304_08159_b200 import synth
    dims = (32, 32)
    L = synth.coeff_spheres(dims, [[12.0, 16.0]], [5.0], np.float64)
    rng = np.random.default_rng(7)
    o = oracle_mod.Oracle(dims, np.float64)
    o.set_coeff(L)
    u = rng.standard_normal((2, 32, 32)) * L
    b = o.divergence(u)
    p1, h1, n1, rc1 = o.solve(np.zeros_like(b), b, 1e-8, 200)
    p2, h2, n2, rc2 = o.solve_pcg(np.zeros_like(b), b, 1e-8, 200)
    assert rc1 == 0 and rc2 == 0 and n2 < n1
    A = incidence_laplacian(dims, L)
    live = (-np.diag(A) > 0).reshape(b.shape)
    d = (p1 - p2)[live]
    assert np.abs(d - d.mean()).max() <= 1e-5 * np.abs(p1[live]).max()   # both stop at 1e-8·||b||: error <~ cond(A)·1e-8
    _, rn = o.residual(p2, b)
    assert rn <= 1.01e-8 * np.abs(b).max()                            # the recurrence residual tracks the true one


def test_pcg_bookkeeping(oracle_mod):
    """hist[0] = ||b - A p0||inf; the stop rule multiplies ||b||inf (as SOLVE's: BJ "until ||r||inf <= 1e-4·||b||inf");
    an input that already meets it runs zero iterations and only loses its mean."""
    from paper_2304_08159_b200 import synth
    cfg = synth.make_config(0)
    o = oracle_mod.Oracle(cfg["dims"], np.float32)
    o.set_coeff(cfg["L"])
    b = o.divergence(cfg["u"])
    p, hist, nit, rc = o.solve_pcg(np.zeros_like(b), b, 1e-4, 64)
    assert rc == 0 and 3 < nit < 26 and hist[0] == np.abs(b).max() and hist[-1] <= 1e-4 * hist[0] < hist[-2]
    pc, histc, ncyc, rcc = o.solve(np.zeros_like(b), b, 1e-4, 64)
    assert nit < ncyc
    _, rn = o.residual(p, b)
    assert abs(rn / hist[-1] - 1.0) <= 5e-2                           # fp32 recurrence vs true residual at 1e-4·||b||
    p3, hist3, nit3, rc3 = o.solve_pcg(p + np.float32(0.5), b, 2e-4, 64)
    assert nit3 == 0 and rc3 == 0 and np.abs(p3 - p).max() <= 1e-6 * np.abs(p).max()
    p4, hist4, nit4, rc4 = o.solve_pcg(np.zeros_like(b), b, 0.0, 5)
    assert nit4 == 5 and rc4 == 1 and np.array_equal(hist4, hist[:6])
