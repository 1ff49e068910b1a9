// wl_common.cuh — grid descriptor, reductions, small device helpers shared by all kernels.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace wl {

// Plain-old-data grid descriptor passed by value to kernels.
struct Grid {
    int n;            // 2 or 3
    int N0, N1, N2;   // N2 = 1 in 2-D
    long long M;      // cells
};

__host__ __device__ inline long long cell_index(const Grid& g, int i0, int i1, int i2) {
    return (long long)i0 + (long long)g.N0 * ((long long)i1 + (long long)g.N1 * (long long)i2);
}

// Device-side scalars of one context (one allocation, zeroed/reset by kernels, mirrored to pinned host memory).
struct Scalars {
    unsigned long long absmax_bits[4];  // slot 0: ||b||inf, 1: ||r||inf, 2..3 scratch (bit pattern of a non-negative double)
    double sum_p;                       // sum of p (ordered second stage)
    double mean_p;                      // sum_p / M
    double shift;                       // deferred mean removal: what the next level-0 DOWN kernel subtracts from p on load
    double nb;                          // ||b||inf
    double tol;                         // stop tolerance of the running solve
    int cycle;                          // cycles completed in the running solve
    int done;                           // 1 once hist[cycle] <= tol * nb
    int maxcycles;
    unsigned int ticket;                // CTAs of the running level-0 launch that have finished (last one does the bookkeeping)
    double rho, alpha, beta;            // conjugate-gradient scalars (wl_pcg.cuh)
    int breakdown;                      // rho' = 0 or sigma = 0: the residual is exactly 0
    int pad;
};

// Programmatic dependent launch (sm_90+): `launch_dependents` lets the next kernel of the stream / graph start its prologue
// while this grid is still running; `wait` blocks until every prerequisite grid has completed and its writes are visible.
// Both are no-ops for a kernel launched without the programmatic-serialization attribute.
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

template <typename T> struct Omega;
template <> struct Omega<float> { __host__ __device__ static constexpr float value() { return (float)(2.0 / 3.0); } };
template <> struct Omega<double> { __host__ __device__ static constexpr double value() { return 2.0 / 3.0; } };

// max of non-negative values that does NOT drop a NaN (fmax does): a NaN operand wins, so that a non-finite field shows
// in the norm instead of reading as "converged".
__device__ __forceinline__ double nanmax(double m, double a) { return (a != a || m != m) ? (m + a) : fmax(m, a); }
// max over a warp / CTA of non-negative values, then one atomicMax on the bit pattern (exact, order-free:
// the IEEE bit pattern of non-negative doubles is monotone in the value, Inf and NaN above every finite one).
__device__ __forceinline__ double warp_max(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = nanmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// CTA-wide max of non-negative values; result valid in thread 0.  `red` = 32 doubles of shared memory.
__device__ __forceinline__ double block_max(double v, double* red) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
    v = warp_max(v);
    if (lane == 0) red[w] = v;
    __syncthreads();
    if (w == 0) {
        v = (lane < nw) ? red[lane] : 0.0;
        v = warp_max(v);
    }
    __syncthreads();
    return v;
}
__device__ __forceinline__ double block_sum(double v, double* red) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
    v = warp_sum(v);
    if (lane == 0) red[w] = v;
    __syncthreads();
    if (w == 0) {
        v = (lane < nw) ? red[lane] : 0.0;
        v = warp_sum(v);
    }
    __syncthreads();
    return v;
}

__device__ __forceinline__ void atomic_max_nonneg(unsigned long long* slot, double v) {
    atomicMax(slot, (unsigned long long)__double_as_longlong(fabs(v)));   // fabs: a NaN with the sign bit set still sorts on top
}

// ---- solve bookkeeping of the lagged stop test, run by the LAST CTA of the level-0 launches -------------
// After the level-0 DOWN launch g of a solve: slot 1 holds ||b - A p_k||inf of its INPUT p_k (k = g-1 cycles done; k = 0: the
// caller's initial guess).  Record it as hist[k], take the stop decision, mirror to the pinned host copy, clear the slot for
// the next launch.  When it stops, every later kernel of this and of the next (already enqueued) launch returns at once
// (check_done) and p still holds p_k: the DOWN kernel writes scratch only.  One thread.
__device__ __forceinline__ void solve_check_lagged(Scalars* scal, double* __restrict__ hist, Scalars* host_mirror,
                                                   double* host_hist) {
    const int k = scal->cycle;
    const double r = __longlong_as_double((long long)scal->absmax_bits[1]);
    scal->absmax_bits[1] = 0ULL;
    if (k > scal->maxcycles) return;   // cannot happen inside a solve (done is set at k = maxcycles); keeps stand-alone launches in bounds
    hist[k] = r;
    if (!(r > scal->tol * scal->nb) || k >= scal->maxcycles) scal->done = 1;
    host_hist[k] = r;
    host_mirror->nb = scal->nb;
    __threadfence_system();
    *((volatile int*)&host_mirror->cycle) = k + 1;   // number of history entries the host may read
}
// After the level-0 UP launch: mean_p = (sum of the per-CTA partials in a FIXED order) / M — lane l adds partials l, l+32,
// ... in sequence, a shuffle tree combines the 32 lane sums: the same order on every run (bit-reproducible) — then the
// cycle counter and the shift the next DOWN launch subtracts on load.  One warp (all 32 lanes must call).
__device__ __forceinline__ void solve_finish_mean_lagged(Scalars* scal, const double* partials, int nparts, long long M) {
    const int lane = threadIdx.x & 31;
    double s = 0.0;
    for (int i = lane; i < nparts; i += 32) s += ((const volatile double*)partials)[i];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
    if (lane == 0) {
        scal->sum_p = s;
        scal->mean_p = s / (double)M;
        scal->cycle += 1;
        scal->shift = scal->mean_p;
    }
}

// ordered sum of nparts partials with stride `stride` doubles, by one warp (lane l adds l, l+32, ...; shuffle tree)
__device__ __forceinline__ double ordered_sum(const double* partials, int nparts, int stride) {
    const int lane = threadIdx.x & 31;
    double s = 0.0;
    for (int i = lane; i < nparts; i += 32) s += ((const volatile double*)partials)[(size_t)i * stride];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
    return __shfl_sync(0xffffffffu, s, 0);
}

// Conjugate-gradient bookkeeping after z = V(r) (wl_pcg.cuh): partials hold per-CTA (sum z, sum r z) pairs; mean of z, beta =
// rho'/rho (0 on the first iteration), rho <- rho'; rho' = 0 ends the solve.  One warp (all 32 lanes must call).
__device__ __forceinline__ void pcg_finish_dot(Scalars* scal, const double* partials, int nparts, long long M) {
    const double tz = ordered_sum(partials, nparts, 2);
    const double trz = ordered_sum(partials + 1, nparts, 2);
    if ((threadIdx.x & 31) == 0) {
        scal->mean_p = tz / (double)M;                       // mz
        scal->beta = (scal->cycle == 0 || scal->rho == 0.0) ? 0.0 : trz / scal->rho;
        scal->rho = trz;
        if (trz == 0.0) scal->breakdown = 1;
    }
}

}  // namespace wl
