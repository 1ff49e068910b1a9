// wl_generic.cuh — one straightforward kernel per step of the path, for ANY grid shape (N_i >= 4, 2-D or 3-D,
// fp32 or fp64).  They are the library's any-shape path (odd extents, tiny levels) and the A/B reference for
// the fused kernels in wl_fused.cuh.  One thread per cell, grid-stride, unit-stride axis across the warp.
//
// Arithmetic follows the operator as BASELINE.json north_star states it ("Problem statement"):
//   (A x)_I = sum_i [ L[i][I+d_i] (x[I+d_i]-x[I]) + L[i][I] (x[I-d_i]-x[I]) ],  walls have L = 0 and are never read.
#pragma once
#include "wl_common.cuh"

namespace wl {

template <typename T, int ND>
__device__ __forceinline__ void decompose(const Grid& g, long long I, int& i0, int& i1, int& i2) {
    long long q = I / g.N0;
    i0 = (int)(I - q * g.N0);
    if (ND == 3) {
        long long q2 = q / g.N1;
        i1 = (int)(q - q2 * g.N1);
        i2 = (int)q2;
    } else {
        i1 = (int)q;
        i2 = 0;
    }
}

// A x and D = -diag(A) at one cell.
template <typename T, int ND>
__device__ __forceinline__ void stencil_cell(const Grid& g, const T* __restrict__ L, const T* __restrict__ x,
                                             long long I, int i0, int i1, int i2, T& Ax, T& D) {
    const int Ii[3] = {i0, i1, i2};
    const int Ni[3] = {g.N0, g.N1, g.N2};
    const long long st[3] = {1, (long long)g.N0, (long long)g.N0 * g.N1};
    const T xc = x[I];
    T s = 0, d = 0;
#pragma unroll
    for (int i = 0; i < ND; ++i) {
        const T* Li = L + (long long)i * g.M;
        T Lp = 0, Lm = 0;
        if (Ii[i] + 1 < Ni[i]) {
            Lp = Li[I + st[i]];
            s += Lp * (x[I + st[i]] - xc);
        }
        if (Ii[i] > 0) {
            Lm = Li[I];
            s += Lm * (x[I - st[i]] - xc);
        }
        d += Lm + Lp;
    }
    Ax = s;
    D = d;
}

// H0 level 0: copy the caller's L, forcing the stored wall plane I_i = 0 of component i to 0.
template <typename T, int ND>
__global__ void k_copy_coeff(Grid g, const T* __restrict__ Lin, T* __restrict__ Lout) {
    const long long total = g.M * ND;
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(e / g.M);
        const long long I = e - (long long)i * g.M;
        int i0, i1, i2;
        decompose<T, ND>(g, I, i0, i1, i2);
        const int Ii[3] = {i0, i1, i2};
        Lout[e] = (Ii[i] == 0) ? (T)0 : Lin[e];
    }
}

// H0 level l -> l+1: Lc[i][J] = sum of the 2^(n-1) fine faces of direction i in coarse face (J,i), fixed tree
// (tangential axes j < k: (00 + 10) + (01 + 11)) — bit-exact against the oracle.  __fadd_rn-style plain adds: no
// FMA can be formed from additions alone, so the compiler cannot change the result.
template <typename T, int ND>
__global__ void k_coarsen(Grid gf, Grid gc, const T* __restrict__ Lf, T* __restrict__ Lc) {
    const long long total = gc.M * ND;
    const long long st[3] = {1, (long long)gf.N0, (long long)gf.N0 * gf.N1};
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(e / gc.M);
        const long long J = e - (long long)i * gc.M;
        int j0, j1, j2;
        decompose<T, ND>(gc, J, j0, j1, j2);
        const long long base = 2LL * j0 + st[1] * (2LL * j1) + (ND == 3 ? st[2] * (2LL * j2) : 0);
        const T* Lfi = Lf + (long long)i * gf.M;
        const int tj = (i == 0) ? 1 : 0;
        T s;
        if (ND == 2) {
            s = Lfi[base] + Lfi[base + st[tj]];
        } else {
            const int tk = (i == 2) ? 1 : 2;
            const T a0 = Lfi[base] + Lfi[base + st[tj]];
            const T a1 = Lfi[base + st[tk]] + Lfi[base + st[tj] + st[tk]];
            s = a0 + a1;
        }
        Lc[e] = s;
    }
}

// H1: b[I] = sum_i (u[i][I+d_i] - u[i][I]); unstored upper wall face = 0.  All n directions in one kernel.
template <typename T, int ND>
__global__ void k_divergence(Grid g, const T* __restrict__ u, T* __restrict__ b) {
    const int Ni[3] = {g.N0, g.N1, g.N2};
    const long long st[3] = {1, (long long)g.N0, (long long)g.N0 * g.N1};
    for (long long I = (long long)blockIdx.x * blockDim.x + threadIdx.x; I < g.M; I += (long long)gridDim.x * blockDim.x) {
        int i0, i1, i2;
        decompose<T, ND>(g, I, i0, i1, i2);
        const int Ii[3] = {i0, i1, i2};
        T s = 0;
#pragma unroll
        for (int i = 0; i < ND; ++i) {
            const T* ui = u + (long long)i * g.M;
            const T up = (Ii[i] + 1 < Ni[i]) ? ui[I + st[i]] : (T)0;
            s += up - ui[I];
        }
        b[I] = s;
    }
}

// H8: u[i][I] -= L[i][I] (p[I] - p[I-d_i]) for all i in one kernel; plane I_i = 0 untouched.
template <typename T, int ND>
__global__ void k_gradient(Grid g, const T* __restrict__ L, T* __restrict__ u, const T* __restrict__ p) {
    const long long st[3] = {1, (long long)g.N0, (long long)g.N0 * g.N1};
    for (long long I = (long long)blockIdx.x * blockDim.x + threadIdx.x; I < g.M; I += (long long)gridDim.x * blockDim.x) {
        int i0, i1, i2;
        decompose<T, ND>(g, I, i0, i1, i2);
        const int Ii[3] = {i0, i1, i2};
        const T pc = p[I];
#pragma unroll
        for (int i = 0; i < ND; ++i) {
            if (Ii[i] > 0) {
                const long long e = (long long)i * g.M + I;
                u[e] -= L[e] * (pc - p[I - st[i]]);
            }
        }
    }
}

// H3: one damped-Jacobi sweep, out of place.  `shift` (nullable) is subtracted from the input on the fly
// (deferred mean removal of the previous cycle: x_in - (T)mean is exactly what the oracle smooths).
template <typename T, int ND>
__global__ void k_jacobi(Grid g, const T* __restrict__ L, const T* __restrict__ xin, const T* __restrict__ b,
                         T* __restrict__ xout) {
    const T omega = Omega<T>::value();
    for (long long I = (long long)blockIdx.x * blockDim.x + threadIdx.x; I < g.M; I += (long long)gridDim.x * blockDim.x) {
        int i0, i1, i2;
        decompose<T, ND>(g, I, i0, i1, i2);
        T Ax, D;
        stencil_cell<T, ND>(g, L, xin, I, i0, i1, i2, Ax, D);
        const T invD = (D > (T)0) ? (T)1 / D : (T)0;
        xout[I] = xin[I] + omega * invD * (Ax - b[I]);
    }
}

// First sweep from x = 0 (coarse levels): x_out = 0 + w invD (0 - b) — identical to k_jacobi on a zero field.
template <typename T, int ND>
__global__ void k_jacobi_from_zero(Grid g, const T* __restrict__ L, const T* __restrict__ b, T* __restrict__ xout) {
    const T omega = Omega<T>::value();
    const int Ni[3] = {g.N0, g.N1, g.N2};
    const long long st[3] = {1, (long long)g.N0, (long long)g.N0 * g.N1};
    for (long long I = (long long)blockIdx.x * blockDim.x + threadIdx.x; I < g.M; I += (long long)gridDim.x * blockDim.x) {
        int i0, i1, i2;
        decompose<T, ND>(g, I, i0, i1, i2);
        const int Ii[3] = {i0, i1, i2};
        T D = 0;
#pragma unroll
        for (int i = 0; i < ND; ++i) {
            const T* Li = L + (long long)i * g.M;
            const T Lp = (Ii[i] + 1 < Ni[i]) ? Li[I + st[i]] : (T)0;
            const T Lm = (Ii[i] > 0) ? Li[I] : (T)0;
            D += Lm + Lp;
        }
        const T invD = (D > (T)0) ? (T)1 / D : (T)0;
        xout[I] = omega * invD * ((T)0 - b[I]);
    }
}

// H4: bc[J] = sum over children of (b - A x); one thread per COARSE cell, children summed pairwise along axis 0,
// then 1, then 2.  Also zeroes xc (x_{l+1} = 0) when xc != nullptr.
template <typename T, int ND>
__global__ void k_residual_restrict(Grid gf, Grid gc, const T* __restrict__ L, const T* __restrict__ x,
                                    const T* __restrict__ b, T* __restrict__ bc, T* __restrict__ xc) {
    for (long long J = (long long)blockIdx.x * blockDim.x + threadIdx.x; J < gc.M; J += (long long)gridDim.x * blockDim.x) {
        int j0, j1, j2;
        decompose<T, ND>(gc, J, j0, j1, j2);
        T s2[2] = {0, 0};
#pragma unroll
        for (int c2 = 0; c2 < (ND == 3 ? 2 : 1); ++c2) {
            T s1[2];
#pragma unroll
            for (int c1 = 0; c1 < 2; ++c1) {
                T r[2];
#pragma unroll
                for (int c0 = 0; c0 < 2; ++c0) {
                    const int i0 = 2 * j0 + c0, i1 = 2 * j1 + c1, i2 = (ND == 3) ? 2 * j2 + c2 : 0;
                    const long long I = cell_index(gf, i0, i1, i2);
                    T Ax, D;
                    stencil_cell<T, ND>(gf, L, x, I, i0, i1, i2, Ax, D);
                    r[c0] = b[I] - Ax;
                }
                s1[c1] = r[0] + r[1];
            }
            s2[c2] = s1[0] + s1[1];
        }
        bc[J] = (ND == 3) ? (s2[0] + s2[1]) : s2[0];
        if (xc) xc[J] = (T)0;
    }
}

// H6 (first half): x[I] += xc[floor(I/2)].
template <typename T, int ND>
__global__ void k_prolong_add(Grid gf, Grid gc, const T* __restrict__ xc, T* __restrict__ x) {
    for (long long I = (long long)blockIdx.x * blockDim.x + threadIdx.x; I < gf.M; I += (long long)gridDim.x * blockDim.x) {
        int i0, i1, i2;
        decompose<T, ND>(gf, I, i0, i1, i2);
        x[I] += xc[cell_index(gc, i0 >> 1, i1 >> 1, i2 >> 1)];
    }
}

// H6 (first half), out of place: xout[I] = xin[I] + xc[floor(I/2)].
template <typename T, int ND>
__global__ void k_prolong_out(Grid gf, Grid gc, const T* __restrict__ xc, const T* __restrict__ xin, T* __restrict__ xout) {
    for (long long I = (long long)blockIdx.x * blockDim.x + threadIdx.x; I < gf.M; I += (long long)gridDim.x * blockDim.x) {
        int i0, i1, i2;
        decompose<T, ND>(gf, I, i0, i1, i2);
        xout[I] = xin[I] + xc[cell_index(gc, i0 >> 1, i1 >> 1, i2 >> 1)];
    }
}

// ||v||inf into scal->absmax_bits[slot] (slot must have been zeroed).
template <typename T>
__global__ void k_absmax(long long M, const T* __restrict__ v, Scalars* scal, int slot) {
    __shared__ double red[32];
    double m = 0.0;
    for (long long I = (long long)blockIdx.x * blockDim.x + threadIdx.x; I < M; I += (long long)gridDim.x * blockDim.x)
        m = nanmax(m, fabs((double)v[I]));
    m = block_max(m, red);
    if (threadIdx.x == 0) atomic_max_nonneg(&scal->absmax_bits[slot], m);
}

// H2/H7: ||b - A p||inf into absmax_bits[slot] and per-CTA partial sums of p into `partials` (one double per CTA).
template <typename T, int ND>
__global__ void k_resnorm_sum(Grid g, const T* __restrict__ L, const T* __restrict__ p, const T* __restrict__ b,
                              Scalars* scal, int slot, double* __restrict__ partials) {
    __shared__ double red[32];
    double m = 0.0, s = 0.0;
    for (long long I = (long long)blockIdx.x * blockDim.x + threadIdx.x; I < g.M; I += (long long)gridDim.x * blockDim.x) {
        int i0, i1, i2;
        decompose<T, ND>(g, I, i0, i1, i2);
        T Ax, D;
        stencil_cell<T, ND>(g, L, p, I, i0, i1, i2, Ax, D);
        m = nanmax(m, fabs((double)(b[I] - Ax)));
        s += (double)p[I];
    }
    m = block_max(m, red);
    s = block_sum(s, red);
    if (threadIdx.x == 0) {
        atomic_max_nonneg(&scal->absmax_bits[slot], m);
        partials[blockIdx.x] = s;
    }
}

// Σp only (per-CTA partials).
template <typename T>
__global__ void k_sum(long long M, const T* __restrict__ p, double* __restrict__ partials) {
    __shared__ double red[32];
    double s = 0.0;
    for (long long I = (long long)blockIdx.x * blockDim.x + threadIdx.x; I < M; I += (long long)gridDim.x * blockDim.x)
        s += (double)p[I];
    s = block_sum(s, red);
    if (threadIdx.x == 0) partials[blockIdx.x] = s;
}

// p -= (T)mean, mean read from the device scalars.
template <typename T>
__global__ void k_shift(long long M, T* __restrict__ p, const Scalars* __restrict__ scal) {
    const T m = (T)scal->mean_p;
    for (long long I = (long long)blockIdx.x * blockDim.x + threadIdx.x; I < M; I += (long long)gridDim.x * blockDim.x)
        p[I] -= m;
}

// ---- single-thread bookkeeping kernels (ordered second stage of the reductions, stop test) ------------------------

// mean_p = (sum of the per-CTA partials in a FIXED order) / M.  One warp: lane l adds partials l, l+32, ... in sequence,
// then a shuffle tree combines the 32 lane sums — the same order on every run (bit-reproducible), 32 independent
// chains instead of one serial chain of global loads.
__global__ void k_finish_mean(Scalars* scal, const double* __restrict__ partials, int nparts, long long M) {
    if (blockIdx.x == 0 && threadIdx.x < 32) {
        double s = 0.0;
        for (int i = threadIdx.x; i < nparts; i += 32) s += partials[i];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
        if (threadIdx.x == 0) {
            scal->sum_p = s;
            scal->mean_p = s / (double)M;
        }
    }
}

// zero an absmax slot
__global__ void k_zero_slot(Scalars* scal, int slot) {
    if (threadIdx.x == 0 && blockIdx.x == 0) scal->absmax_bits[slot] = 0ULL;
}

// solve bookkeeping: init (nb from slot 0, hist[0] from slot 1) and per-cycle record (hist[++cycle] from slot 1)
// (`hist` = device array of maxcycles+1 doubles)
__global__ void k_solve_begin(Scalars* scal, double* __restrict__ hist, double tol, int maxcycles) {
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        scal->nb = __longlong_as_double((long long)scal->absmax_bits[0]);
        const double r0 = __longlong_as_double((long long)scal->absmax_bits[1]);
        hist[0] = r0;
        scal->tol = tol;
        scal->maxcycles = maxcycles;
        scal->cycle = 0;
        scal->shift = 0.0;
        scal->done = (r0 > tol * scal->nb && maxcycles > 0) ? 0 : 1;
    }
}
__global__ void k_cycle_end(Scalars* scal, double* __restrict__ hist, int deferred, Scalars* host_mirror,
                            double* host_hist) {
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        if (scal->done) return;  // a speculative cycle after convergence changes nothing
        scal->shift = deferred ? scal->mean_p : 0.0;  // what the next level-0 DOWN kernel subtracts on load
        const int k = scal->cycle + 1;
        const double r = __longlong_as_double((long long)scal->absmax_bits[1]);
        scal->cycle = k;
        hist[k] = r;
        const int done = (!(r > scal->tol * scal->nb) || k >= scal->maxcycles) ? 1 : 0;
        if (done) scal->done = 1;
        // pinned host mirror (device-mapped): the host polls `cycle` instead of synchronising the stream
        host_hist[k] = r;
        __threadfence_system();
        *((volatile int*)&host_mirror->cycle) = k;
    }
}

// Lagged solve (the stop test rides on the level-0 launches: solve_check_lagged / solve_finish_mean_lagged in wl_common.cuh):
// nb from slot 0 (||b||inf), nothing else is known yet; slot 1 and the CTA ticket start at 0.
__global__ void k_solve_begin_lagged(Scalars* scal, double tol, int maxcycles) {
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        scal->nb = __longlong_as_double((long long)scal->absmax_bits[0]);
        scal->absmax_bits[1] = 0ULL;
        scal->ticket = 0u;
        scal->tol = tol;
        scal->maxcycles = maxcycles;
        scal->cycle = 0;
        scal->shift = 0.0;
        scal->done = 0;
    }
}
}  // namespace wl
