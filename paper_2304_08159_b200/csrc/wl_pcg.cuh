// wl_pcg.cuh — level-0 vector kernels of the V-cycle-preconditioned conjugate-gradient solve (
// PAPER.md:38 "we now use Conjugate-Gradient smoothing within the GMG levels"; DESIGN.md §3 reading 13).
//
//   r = b - A x;  repeat:  z = V(r)  [one V-cycle from z = 0: the fused kernels of wl_fused*.cuh];
//   rho' = r·z, mz = mean(z);  beta = rho'/rho;  p = (z - mz) + beta p;  q = A p;  sigma = p·q;  alpha = rho'/sigma;
//   x += alpha p;  r -= alpha q;  hist[k] = ||r||inf.
//
// Every reduction is a per-CTA fp64 partial + an ordered second stage run by the LAST CTA of the same launch (ticket), so
// an iteration has no single-thread kernels and is bit-reproducible from run to run.  Dot products accumulate in fp64
// (products of two T values are exact in fp64 for T = float), the scalars are formed in fp64 and cast to T, the vector
// updates round every multiply and add separately (no FMA): the oracle's arithmetic.
#pragma once
#include "wl_common.cuh"
#include "wl_generic.cuh"

namespace wl {

// ordered sum of nparts partials with stride `stride` doubles, by one warp (lane l adds l, l+32, ...; shuffle tree)
__device__ __forceinline__ double ordered_sum(const double* partials, int nparts, int stride) {
    const int lane = threadIdx.x & 31;
    double s = 0.0;
    for (int i = lane; i < nparts; i += 32) s += ((const volatile double*)partials)[(size_t)i * stride];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
    return __shfl_sync(0xffffffffu, s, 0);
}

// true in every thread of the last CTA of the launch to get here (after publishing its partials), false elsewhere
__device__ __forceinline__ bool last_cta(Scalars* scal) {
    __shared__ int s_last;
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        const unsigned int ticket = atomicAdd(&scal->ticket, 1u);
        s_last = (ticket == gridDim.x - 1) ? 1 : 0;
        if (s_last) scal->ticket = 0u;
    }
    __syncthreads();
    if (s_last) __threadfence();
    return s_last != 0;
}

// record hist[k] = ||r||inf (slot 1), take the stop decision, mirror to the host (one thread)
__device__ __forceinline__ void pcg_record(Scalars* scal, double* hist, Scalars* host_mirror, double* host_hist) {
    const int k = scal->cycle;
    const double r = __longlong_as_double((long long)scal->absmax_bits[1]);
    scal->absmax_bits[1] = 0ULL;
    if (k > scal->maxcycles) return;
    hist[k] = r;
    if (!(r > scal->tol * scal->nb) || k >= scal->maxcycles) scal->done = 1;
    host_hist[k] = r;
    host_mirror->nb = scal->nb;
    host_mirror->done = scal->done;
    __threadfence_system();
    *((volatile int*)&host_mirror->cycle) = k + 1;   // number of history entries the host may read
}

__global__ void k_pcg_begin(Scalars* scal, double tol, int maxit) {
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        scal->nb = __longlong_as_double((long long)scal->absmax_bits[0]);
        scal->absmax_bits[1] = 0ULL;
        scal->ticket = 0u;
        scal->tol = tol;
        scal->maxcycles = maxit;
        scal->cycle = 0;
        scal->shift = 0.0;
        scal->done = 0;
        scal->rho = 0.0;
    }
}

// r = b - A x, ||r||inf -> hist[0] and the first stop decision
template <typename T, int ND>
__global__ void k_pcg_residual(Grid g, const T* __restrict__ L, const T* __restrict__ x, const T* __restrict__ b,
                               T* __restrict__ r, Scalars* scal, double* hist, Scalars* host_mirror, double* host_hist) {
    __shared__ double red[32];
    double m = 0.0;
    for (long long I = (long long)blockIdx.x * blockDim.x + threadIdx.x; I < g.M; I += (long long)gridDim.x * blockDim.x) {
        int i0, i1, i2;
        decompose<T, ND>(g, I, i0, i1, i2);
        T Ax, D;
        stencil_cell<T, ND>(g, L, x, I, i0, i1, i2, Ax, D);
        const T rv = b[I] - Ax;
        r[I] = rv;
        m = nanmax(m, fabs((double)rv));
    }
    m = block_max(m, red);
    if (threadIdx.x == 0) atomic_max_nonneg(&scal->absmax_bits[1], m);
    if (last_cta(scal) && threadIdx.x == 0) pcg_record(scal, hist, host_mirror, host_hist);
}

// rho' = sum r z, mz = mean z (z as the V-cycle left it); beta = rho'/rho (0 on the first iteration); rho' = 0 ends the solve
template <typename T>
__global__ void k_pcg_dot_rz(long long M, const T* __restrict__ r, const T* __restrict__ z, Scalars* scal,
                             double* __restrict__ partials) {
    if (scal->done) return;
    __shared__ double red[32];
    double sz = 0.0, srz = 0.0;
    for (long long I = (long long)blockIdx.x * blockDim.x + threadIdx.x; I < M; I += (long long)gridDim.x * blockDim.x) {
        const double zv = (double)z[I];
        sz += zv;
        srz += (double)r[I] * zv;
    }
    sz = block_sum(sz, red);
    srz = block_sum(srz, red);
    if (threadIdx.x == 0) { partials[2 * blockIdx.x] = sz; partials[2 * blockIdx.x + 1] = srz; }
    if (last_cta(scal) && threadIdx.x < 32) {
        const double tz = ordered_sum(partials, (int)gridDim.x, 2);
        const double trz = ordered_sum(partials + 1, (int)gridDim.x, 2);
        if (threadIdx.x == 0) {
            scal->mean_p = tz / (double)M;                       // mz
            scal->beta = (scal->cycle == 0 || scal->rho == 0.0) ? 0.0 : trz / scal->rho;
            scal->rho = trz;
            if (trz == 0.0) scal->breakdown = 1;
        }
    }
}

// p = (z - mz) + beta p
template <typename T>
__global__ void k_pcg_update_p(long long M, const T* __restrict__ z, T* __restrict__ p, const Scalars* __restrict__ scal) {
    if (scal->done || scal->breakdown) return;
    const T mz = (T)scal->mean_p, beta = (T)scal->beta;
    for (long long I = (long long)blockIdx.x * blockDim.x + threadIdx.x; I < M; I += (long long)gridDim.x * blockDim.x) {
        const T zs = z[I] - mz;
        const T bp = beta * p[I];
        p[I] = zs + bp;
    }
}

// q = A p, sigma = sum p q; alpha = rho / sigma
template <typename T, int ND>
__global__ void k_pcg_Ap(Grid g, const T* __restrict__ L, const T* __restrict__ p, T* __restrict__ q, Scalars* scal,
                         double* __restrict__ partials) {
    if (scal->done || scal->breakdown) return;
    __shared__ double red[32];
    double s = 0.0;
    for (long long I = (long long)blockIdx.x * blockDim.x + threadIdx.x; I < g.M; I += (long long)gridDim.x * blockDim.x) {
        int i0, i1, i2;
        decompose<T, ND>(g, I, i0, i1, i2);
        T Ax, D;
        stencil_cell<T, ND>(g, L, p, I, i0, i1, i2, Ax, D);
        q[I] = Ax;
        s += (double)p[I] * (double)Ax;
    }
    s = block_sum(s, red);
    if (threadIdx.x == 0) partials[blockIdx.x] = s;
    if (last_cta(scal) && threadIdx.x < 32) {
        const double sigma = ordered_sum(partials, (int)gridDim.x, 1);
        if (threadIdx.x == 0) {
            if (sigma == 0.0) scal->breakdown = 1;
            else scal->alpha = scal->rho / sigma;
        }
    }
}

// x += alpha p, r -= alpha q, ||r||inf -> hist[k+1], stop decision.  A breakdown (rho' = 0 or sigma = 0: nothing left to
// correct) ends the solve as converged without touching x.
template <typename T>
__global__ void k_pcg_update_xr(long long M, T* __restrict__ x, T* __restrict__ r, const T* __restrict__ p,
                                const T* __restrict__ q, Scalars* scal, double* hist, Scalars* host_mirror, double* host_hist) {
    if (scal->done) return;
    __shared__ double red[32];
    const bool brk = scal->breakdown != 0;
    double m = 0.0;
    if (!brk) {
        const T alpha = (T)scal->alpha;
        for (long long I = (long long)blockIdx.x * blockDim.x + threadIdx.x; I < M; I += (long long)gridDim.x * blockDim.x) {
            const T ap = alpha * p[I];
            x[I] = x[I] + ap;
            const T aq = alpha * q[I];
            const T rv = r[I] - aq;
            r[I] = rv;
            m = nanmax(m, fabs((double)rv));
        }
    }
    m = block_max(m, red);
    if (threadIdx.x == 0 && !brk) atomic_max_nonneg(&scal->absmax_bits[1], m);
    if (last_cta(scal) && threadIdx.x == 0) {
        if (brk) {
            scal->done = 1;
            host_mirror->done = 2;
            __threadfence_system();
            *((volatile int*)&host_mirror->cycle) = scal->cycle + 2;   // wakes the host without a new history entry
        } else {
            scal->cycle += 1;
            pcg_record(scal, hist, host_mirror, host_hist);
        }
    }
}

}  // namespace wl
