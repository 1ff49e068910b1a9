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
#include "wl_rows.cuh"

namespace wl {

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
        scal->breakdown = 0;   // a breakdown of an earlier solve (e.g. an all-solid field, z = 0) must not end this one
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
    if (last_cta(scal) && threadIdx.x < 32) pcg_finish_dot(scal, partials, (int)gridDim.x, M);
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

// the same with 16-byte accesses (M a multiple of the vector width, aligned arrays)
template <typename T>
__global__ void k_pcg_update_p_vec(long long M, const T* __restrict__ z, T* __restrict__ p, const Scalars* __restrict__ scal) {
    if (scal->done || scal->breakdown) return;
    constexpr int VEC = 16 / (int)sizeof(T);
    const T mz = (T)scal->mean_p, beta = (T)scal->beta;
    const long long nv = M / VEC;
    for (long long v = (long long)blockIdx.x * blockDim.x + threadIdx.x; v < nv; v += (long long)gridDim.x * blockDim.x) {
        T zv[VEC], pv[VEC];
        ld_vec<T, VEC>(z + v * VEC, zv);
        ld_vec<T, VEC>(p + v * VEC, pv);
#pragma unroll
        for (int k = 0; k < VEC; ++k) {
            const T zs = zv[k] - mz;
            const T bp = beta * pv[k];
            pv[k] = zs + bp;
        }
        st_vec<T, VEC>(p + v * VEC, pv);
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

// The same as a row kernel (16-byte loads along the unit-stride axis, two integer divisions per row instead of per cell; rows
// of whole vectors, aligned arrays).  Per cell the terms and their order are stencil_cell's: upper face, lower face; axis 0, 1, 2.
// RESID: q = b - A p and ||q||inf -> hist[0] with the first stop decision (k_pcg_residual) instead of q = A p, sigma, alpha.
template <typename T, int ND, bool RESID>
__global__ void __launch_bounds__(kRowsX* kRowsY) k_pcg_Ap_rows(Grid g, const T* __restrict__ L, const T* __restrict__ p,
                                                               T* __restrict__ q, Scalars* scal, double* __restrict__ partials,
                                                               const T* __restrict__ b, double* hist, Scalars* host_mirror,
                                                               double* host_hist) {
    if (!RESID && (scal->done || scal->breakdown)) return;
    constexpr int VEC = 16 / (int)sizeof(T);
    __shared__ double red[32];
    const int nvx = g.N0 / VEC;
    const long long nrows = (long long)g.N1 * g.N2;
    const long long sy = g.N0, sz = (long long)g.N0 * g.N1;
    const T* L0 = L;
    const T* L1 = L + g.M;
    const T* L2 = L + 2 * g.M;
    double s = 0.0;
    for (long long r = (long long)blockIdx.x * kRowsY + threadIdx.y; r < nrows; r += (long long)gridDim.x * kRowsY) {
        const int z = (int)(r / g.N1), y = (int)(r - (long long)z * g.N1);
        const bool up1 = y + 1 < g.N1, lo1 = y > 0, up2 = (ND == 3) && (z + 1 < g.N2), lo2 = (ND == 3) && (z > 0);
        for (int vx = threadIdx.x; vx < nvx; vx += kRowsX) {
            const int x = vx * VEC;
            const long long e0 = r * g.N0 + x;
            T pc[VEC], l0[VEC], l1[VEC], l1u[VEC], py_u[VEC], py_l[VEC], out[VEC];
            ld_vec<T, VEC>(p + e0, pc);
            ld_vec<T, VEC>(L0 + e0, l0);
            ld_vec<T, VEC>(L1 + e0, l1);
            T bv[VEC];
            if (RESID) ld_vec<T, VEC>(b + e0, bv);
            const bool upx = x + VEC < g.N0;
            const T pxn = upx ? p[e0 + VEC] : (T)0, l0n = upx ? L0[e0 + VEC] : (T)0;
            const T pxm = (x > 0) ? p[e0 - 1] : (T)0;
            if (up1) { ld_vec<T, VEC>(p + e0 + sy, py_u); ld_vec<T, VEC>(L1 + e0 + sy, l1u); }
            if (lo1) ld_vec<T, VEC>(p + e0 - sy, py_l);
            T l2[VEC], l2u[VEC], pz_u[VEC], pz_l[VEC];
            if (ND == 3) {
                ld_vec<T, VEC>(L2 + e0, l2);
                if (up2) { ld_vec<T, VEC>(p + e0 + sz, pz_u); ld_vec<T, VEC>(L2 + e0 + sz, l2u); }
                if (lo2) ld_vec<T, VEC>(p + e0 - sz, pz_l);
            }
#pragma unroll
            for (int k = 0; k < VEC; ++k) {
                const T xc = pc[k];
                T a = 0;
                if (k + 1 < VEC) a += l0[(k + 1) % VEC] * (pc[(k + 1) % VEC] - xc);
                else if (upx) a += l0n * (pxn - xc);
                if (k > 0) a += l0[k] * (pc[(k + VEC - 1) % VEC] - xc);
                else if (x > 0) a += l0[k] * (pxm - xc);
                if (up1) a += l1u[k] * (py_u[k] - xc);
                if (lo1) a += l1[k] * (py_l[k] - xc);
                if (ND == 3) {
                    if (up2) a += l2u[k] * (pz_u[k] - xc);
                    if (lo2) a += l2[k] * (pz_l[k] - xc);
                }
                if (RESID) {
                    out[k] = bv[k] - a;
                    s = nanmax(s, fabs((double)out[k]));
                } else {
                    out[k] = a;
                    s += (double)xc * (double)a;
                }
            }
            st_vec<T, VEC>(q + e0, out);
        }
    }
    {   // CTA sum (thread index is two-dimensional here), partial, ordered second stage by the last CTA
        const int tid = threadIdx.y * kRowsX + threadIdx.x;
        s = RESID ? warp_max(s) : warp_sum(s);
        if ((tid & 31) == 0) red[tid >> 5] = s;
        __syncthreads();
        if (tid < 32) {
            s = (tid < (kRowsX * kRowsY) / 32) ? red[tid] : 0.0;
            s = RESID ? warp_max(s) : warp_sum(s);
            if (tid == 0) {
                if (RESID) atomic_max_nonneg(&scal->absmax_bits[1], s);
                else partials[blockIdx.x] = s;
            }
        }
    }
    __shared__ int s_last;
    __syncthreads();
    const int tid = threadIdx.y * kRowsX + threadIdx.x;
    if (tid == 0) {
        __threadfence();
        const unsigned int ticket = atomicAdd(&scal->ticket, 1u);
        s_last = (ticket == gridDim.x - 1) ? 1 : 0;
        if (s_last) scal->ticket = 0u;
    }
    __syncthreads();
    if (RESID) {
        if (s_last && tid == 0) { __threadfence(); pcg_record(scal, hist, host_mirror, host_hist); }
    } else if (s_last && tid < 32) {
        __threadfence();
        const double sigma = ordered_sum(partials, (int)gridDim.x, 1);
        if (tid == 0) {
            if (sigma == 0.0) scal->breakdown = 1;
            else scal->alpha = scal->rho / sigma;
        }
    }
}

// x += alpha p, r -= alpha q, ||r||inf -> hist[k+1], stop decision.  A breakdown (rho' = 0 or sigma = 0: nothing left to
// correct) ends the solve as converged without touching x.
template <typename T, bool VECTOR>
__global__ void k_pcg_update_xr(long long M, T* __restrict__ x, T* __restrict__ r, const T* __restrict__ p,
                                const T* __restrict__ q, Scalars* scal, double* hist, Scalars* host_mirror, double* host_hist) {
    if (scal->done) return;
    __shared__ double red[32];
    const bool brk = scal->breakdown != 0;
    double m = 0.0;
    if (!brk) {
        const T alpha = (T)scal->alpha;
        if (VECTOR) {   // 16-byte accesses (M a multiple of the vector width, aligned arrays)
            constexpr int VEC = 16 / (int)sizeof(T);
            const long long nv = M / VEC;
            for (long long v = (long long)blockIdx.x * blockDim.x + threadIdx.x; v < nv; v += (long long)gridDim.x * blockDim.x) {
                T xv[VEC], rv[VEC], pv[VEC], qv[VEC];
                ld_vec<T, VEC>(x + v * VEC, xv);
                ld_vec<T, VEC>(p + v * VEC, pv);
                ld_vec<T, VEC>(r + v * VEC, rv);
                ld_vec<T, VEC>(q + v * VEC, qv);
#pragma unroll
                for (int k = 0; k < VEC; ++k) {
                    const T ap = alpha * pv[k];
                    xv[k] = xv[k] + ap;
                    const T aq = alpha * qv[k];
                    rv[k] = rv[k] - aq;
                    m = nanmax(m, fabs((double)rv[k]));
                }
                st_vec<T, VEC>(x + v * VEC, xv);
                st_vec<T, VEC>(r + v * VEC, rv);
            }
        } else
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
