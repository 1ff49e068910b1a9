"""Independent dense constructions used to pin the oracle.  Nothing here calls the oracle or the CUDA path."""
import numpy as np


# ---------------------------------------------------------------------------------------------
# Independent dense constructions used to pin the oracle (NumPy/SciPy only; nothing below calls
# the oracle).  Cell linear index = I_0 + N_0 (I_1 + N_1 I_2); a cell field of NumPy shape
# (N_{n-1},…,N_0) flattens (C order) to exactly that index.
# ---------------------------------------------------------------------------------------------

def dense_from_apply(apply, M, dtype=np.float64):
    """Dense matrix of a linear map given as a function on flat vectors (columns = images of unit vectors)."""
    A = np.zeros((M, M), dtype=dtype)
    e = np.zeros(M, dtype=dtype)
    for j in range(M):
        e[j] = 1
        A[:, j] = apply(e)
        e[j] = 0
    return A


def incidence_laplacian(dims, L):
    """A = -G^T diag(L) G with G the face-difference (incidence) matrix: row f=(I,i), I_i>=1, has +1 at
    cell I and -1 at cell I-d_i.  Built face by face; independent of the oracle's cell-by-cell stencil form."""
    n = len(dims)
    shape = tuple(reversed(dims))
    M = int(np.prod(dims))
    idx = np.arange(M).reshape(shape)
    A = np.zeros((M, M))
    for i in range(n):
        ax = n - 1 - i
        hi = np.take(idx, np.arange(1, dims[i]), axis=ax).ravel()
        lo = np.take(idx, np.arange(0, dims[i] - 1), axis=ax).ravel()
        w = np.take(np.asarray(L[i], dtype=np.float64), np.arange(1, dims[i]), axis=ax).ravel()
        G = np.zeros((hi.size, M))
        G[np.arange(hi.size), hi] = 1.0
        G[np.arange(hi.size), lo] = -1.0
        A -= G.T @ (w[:, None] * G)
    return A


def restriction_matrix(dims):
    """R (Mc x M): coarse cell J sums fine cells 2J + c, c in {0,1}^n."""
    n = len(dims)
    cd = tuple(d // 2 for d in dims)
    M, Mc = int(np.prod(dims)), int(np.prod(cd))
    fi = np.arange(M).reshape(tuple(reversed(dims)))
    R = np.zeros((Mc, M))
    for I in np.ndindex(*reversed(dims)):  # I in NumPy axis order (I_{n-1},…,I_0)
        J = tuple(v // 2 for v in I)
        Jlin = 0
        for a, v in enumerate(J):  # C-order flatten of shape reversed(cd)
            Jlin = Jlin * cd[n - 1 - a] + v
        R[Jlin, fi[I]] = 1.0
    return R


def random_coeff(dims, rng, dtype=np.float64, dyadic=False):
    n = len(dims)
    shape = (n,) + tuple(reversed(dims))
    if dyadic:
        L = rng.integers(1, 1024, size=shape).astype(np.float64) / 1024.0
    else:
        L = rng.uniform(0.05, 1.0, size=shape)
    for i in range(n):
        sl = [slice(None)] * n
        sl[n - 1 - i] = 0
        L[(i,) + tuple(sl)] = 0.0
    return L.astype(dtype)
