// wl_tail.cuh — the coarse tail of the V-cycle in ONE persistent CTA (H5; BJ "Small coarse levels in a single persistent
// CTA"): every level from `first` down to the coarsest lives in shared memory (x ping-pong, b, L); the CTA walks
// down (2 sweeps, residual, restriction), does the 64 coarsest sweeps, and walks up (injection, 2 sweeps) with
// __syncthreads between steps — no launches, no HBM traffic beyond reading b, L once and writing x once.
// The arithmetic per cell is the generic kernels' (stencil_cell), i.e. the oracle's expression order.
#pragma once
#include "wl_common.cuh"
#include "wl_generic.cuh"

namespace wl {

constexpr int kTailMaxLevels = 8;   // barrier ids 2 .. 2+kTailMaxLevels-1 are used, < 16
constexpr int kTailThreads = 1024;

template <typename T>
struct TailParams {
    int nl;                          // levels in the tail (>= 1); level 0 of the tail = `first` of the hierarchy
    int zero_in;                     // 1: start from x = 0 on the tail's first level; 0: start from x_in
    Grid g[kTailMaxLevels];
    const T* L[kTailMaxLevels];      // global coefficient arrays of each tail level
    unsigned off[kTailMaxLevels];    // byte offset of the level's block in shared memory: xA, xB, b, C, L (ND arrays)
    const T* x_in;                   // tail level 0 initial guess (ignored if zero_in)
    const T* b_in;                   // tail level 0 right-hand side (global)
    T* x_out;                        // tail level 0 result (global)
    int coarsest_is_correction;      // 1: the coarsest level starts from 0 (it is a correction level of the hierarchy)
    const Scalars* scal;             // with check_done: return at once if scal->done (speculative cycle past convergence)
    int check_done;
};

// Named barrier over the first `nthreads` threads of the CTA (a multiple of 32): small levels do not make the whole
// CTA wait.  id 1..15.
__device__ __forceinline__ void bar_sync_n(int id, int nthreads) {
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

// 32-bit index helpers (tail levels have at most a few thousand cells): no 64-bit divisions in the sweeps.
template <int ND>
__device__ __forceinline__ void decompose_i(const Grid& g, int I, int& i0, int& i1, int& i2) {
    // exact for the tail's sizes (I < 2^16, N < 2^10): the float quotient of (I + 1/2) / N is never within rounding
    // error of an integer
    const int q = __float2int_rz(((float)I + 0.5f) * __frcp_rn((float)g.N0));
    i0 = I - q * g.N0;
    if (ND == 3) {
        const int q2 = __float2int_rz(((float)q + 0.5f) * __frcp_rn((float)g.N1));
        i1 = q - q2 * g.N1;
        i2 = q2;
    } else {
        i1 = q;
        i2 = 0;
    }
}
// A x at one cell, the oracle's term order (upper face, lower face; axis 0, 1, 2); absent neighbours are skipped.
template <typename T, int ND>
__device__ __forceinline__ T stencil_i(const Grid& g, const T* L, const T* x, int I, int i0, int i1, int i2) {
    const int Ii[3] = {i0, i1, i2};
    const int Ni[3] = {g.N0, g.N1, g.N2};
    const int st[3] = {1, g.N0, g.N0 * g.N1};
    const int M = (int)g.M;
    const T xc = x[I];
    T s = 0;
#pragma unroll
    for (int i = 0; i < ND; ++i) {
        const T* Li = L + i * M;
        if (Ii[i] + 1 < Ni[i]) s += Li[I + st[i]] * (x[I + st[i]] - xc);
        if (Ii[i] > 0) s += Li[I] * (x[I - st[i]] - xc);
    }
    return s;
}

// One damped-Jacobi sweep over a level held in shared memory; C = omega * invD per cell (precomputed, same rounding as
// the oracle's omega*invD).  Only threads < nthr take part (and synchronise).
template <typename T, int ND>
__device__ __forceinline__ void tail_sweep(const Grid& g, const T* L, const T* C, const T* xin, const T* b, T* xout,
                                           bool from_zero, int nthr) {
    for (int I = threadIdx.x; I < (int)g.M; I += nthr) {
        if (from_zero) {
            xout[I] = C[I] * ((T)0 - b[I]);
        } else {
            int i0, i1, i2;
            decompose_i<ND>(g, I, i0, i1, i2);
            const T Ax = stencil_i<T, ND>(g, L, xin, I, i0, i1, i2);
            xout[I] = xin[I] + C[I] * (Ax - b[I]);
        }
    }
    bar_sync_n(1, nthr);
}

// `sweeps` sweeps on a level with at most one cell per thread (the coarsest level): the cell's coefficients, neighbour
// indices, omega/D and b stay in registers; a sweep is 2*ND shared loads, the stencil, one store and one barrier.
// Starts from XA (or from zero), ping-pongs XA/XB, leaves the result in XA.  sweeps must be even.
template <typename T, int ND>
__device__ __forceinline__ void tail_sweeps_cached(const Grid& g, const T* L, const T* C, T* XA, T* XB, const T* b,
                                                   bool from_zero, int sweeps, int nthr) {
    const int I = threadIdx.x;
    const bool has = I < (int)g.M;
    const int M = (int)g.M;
    T Lf[2 * ND];
    int nb[2 * ND];
    T cI = 0, bI = 0, xv = 0;
    if (has) {
        int i0, i1, i2;
        decompose_i<ND>(g, I, i0, i1, i2);
        const int Ii[3] = {i0, i1, i2};
        const int Ni[3] = {g.N0, g.N1, g.N2};
        const int st[3] = {1, g.N0, g.N0 * g.N1};
#pragma unroll
        for (int i = 0; i < ND; ++i) {
            const bool up = Ii[i] + 1 < Ni[i], lo = Ii[i] > 0;
            nb[2 * i] = up ? I + st[i] : -1;
            nb[2 * i + 1] = lo ? I - st[i] : -1;
            Lf[2 * i] = up ? L[i * M + I + st[i]] : (T)0;
            Lf[2 * i + 1] = lo ? L[i * M + I] : (T)0;
        }
        cI = C[I];
        bI = b[I];
        xv = from_zero ? (T)0 : XA[I];
    } else {
#pragma unroll
        for (int k = 0; k < 2 * ND; ++k) { nb[k] = -1; Lf[k] = (T)0; }
    }
    T* cur = XA;
    T* oth = XB;
    for (int s = 0; s < sweeps; ++s) {
        T xn;
        if (s == 0 && from_zero) {
            xn = cI * ((T)0 - bI);
        } else {
            T a = 0;
#pragma unroll
            for (int k = 0; k < 2 * ND; ++k)
                if (nb[k] >= 0) a += Lf[k] * (cur[nb[k]] - xv);
            xn = xv + cI * (a - bI);
        }
        xv = xn;
        if (has) oth[I] = xn;
        bar_sync_n(1, nthr);
        T* tmp = cur; cur = oth; oth = tmp;
    }
    // an even number of sweeps ends with cur == XA
}

template <typename T, int ND>
__global__ void __launch_bounds__(kTailThreads, 1) k_coarse_tail(TailParams<T> P) {
    pdl_launch_dependents();   // the next kernel of the cycle may set up while the tail runs (it waits before touching data)
    extern __shared__ __align__(16) unsigned char tail_smem[];
    auto XA = [&](int l) -> T* { return (T*)(tail_smem + P.off[l]); };
    auto XB = [&](int l) -> T* { return XA(l) + P.g[l].M; };
    auto B = [&](int l) -> T* { return XA(l) + 2 * P.g[l].M; };
    auto CC = [&](int l) -> T* { return XA(l) + 3 * P.g[l].M; };
    auto LL = [&](int l) -> T* { return XA(l) + 4 * P.g[l].M; };
    const T omega = Omega<T>::value();

    // Stage every level's coefficients in shared memory and derive omega/D from them.  No kernel of a cycle writes the
    // coefficients, so under programmatic dependent launch this part runs while the level above is still draining.
    for (int l = 0; l < P.nl; ++l) {
        const int n = (int)P.g[l].M * ND;
        T* d = LL(l);
        for (int i = threadIdx.x; i < n; i += blockDim.x) d[i] = P.L[l][i];
    }
    __syncthreads();
    for (int l = 0; l < P.nl; ++l) {   // C = omega * invD, D = sum of the cell's face coefficients (oracle order)
        const Grid g = P.g[l];
        const T* L = LL(l);
        T* C = CC(l);
        for (int I = threadIdx.x; I < (int)g.M; I += blockDim.x) {
            int i0, i1, i2;
            decompose_i<ND>(g, I, i0, i1, i2);
            const int Ii[3] = {i0, i1, i2};
            const int Ni[3] = {g.N0, g.N1, g.N2};
            const int st[3] = {1, g.N0, g.N0 * g.N1};
            T D = 0;
#pragma unroll
            for (int i = 0; i < ND; ++i) {
                const T* Li = L + (size_t)i * g.M;
                const T Lp = (Ii[i] + 1 < Ni[i]) ? Li[I + st[i]] : (T)0;
                const T Lm = (Ii[i] > 0) ? Li[I] : (T)0;
                D += Lm + Lp;
            }
            const T invD = (D > (T)0) ? (T)1 / D : (T)0;
            C[I] = omega * invD;
        }
    }
    pdl_wait();                                   // from here on: data the cycle's earlier kernels wrote
    if (P.check_done && P.scal->done) return;     // uniform
    {   // the first level's b (and x)
        const int M = (int)P.g[0].M;
        T* b0 = B(0);
        T* x0 = XA(0);
        for (int i = threadIdx.x; i < M; i += blockDim.x) {
            b0[i] = P.b_in[i];
            if (!P.zero_in) x0[i] = P.x_in[i];
        }
    }
    __syncthreads();

    // threads taking part on a level: enough warps for one cell per thread, at most the CTA
    auto nthr_of = [&](int l) -> int {
        int n = ((int)P.g[l].M + 31) / 32 * 32;
        return n < (int)blockDim.x ? n : (int)blockDim.x;
    };

    const int last = P.nl - 1;
    // ---- down ----------------------------------------------------------------------------------------------------
    for (int l = 0; l < last; ++l) {
        const Grid gf = P.g[l], gc = P.g[l + 1];
        const int nthr = nthr_of(l);
        if ((int)threadIdx.x < nthr) {
            const bool zero = (l > 0) || P.zero_in;
            tail_sweep<T, ND>(gf, LL(l), CC(l), XA(l), B(l), XB(l), zero, nthr);    // XA -> XB
            tail_sweep<T, ND>(gf, LL(l), CC(l), XB(l), B(l), XA(l), false, nthr);   // XB -> XA  (x after 2 pre-sweeps)
            const T* x = XA(l);
            const T* b = B(l);
            const T* L = LL(l);
            T* r = XB(l);                                                           // XB is free: fine residual
            for (int I = threadIdx.x; I < (int)gf.M; I += nthr) {
                int i0, i1, i2;
                decompose_i<ND>(gf, I, i0, i1, i2);
                r[I] = b[I] - stencil_i<T, ND>(gf, L, x, I, i0, i1, i2);
            }
            bar_sync_n(1, nthr);
            T* bc = B(l + 1);
            for (int J = threadIdx.x; J < (int)gc.M; J += nthr) {                   // b_{l+1} = R r: pairwise along 0, 1, 2
                int j0, j1, j2;
                decompose_i<ND>(gc, J, j0, j1, j2);
                T s2[2] = {0, 0};
#pragma unroll
                for (int c2 = 0; c2 < (ND == 3 ? 2 : 1); ++c2) {
                    T s1[2];
#pragma unroll
                    for (int c1 = 0; c1 < 2; ++c1) {
                        const int I = 2 * j0 + gf.N0 * ((2 * j1 + c1) + gf.N1 * ((ND == 3) ? 2 * j2 + c2 : 0));
                        s1[c1] = r[I] + r[I + 1];
                    }
                    s2[c2] = s1[0] + s1[1];
                }
                bc[J] = (ND == 3) ? (s2[0] + s2[1]) : s2[0];
            }
            bar_sync_n(1, nthr);   // also orders this level's threads before the (fewer) threads of the next level
        }
    }
    // ---- coarsest: 64 sweeps, result in XA(last) ---------------------------------------------------------------------
    {
        const Grid g = P.g[last];
        const int nthr = nthr_of(last);
        if ((int)threadIdx.x < nthr) {
            const bool zero = (last > 0) ? true : (P.zero_in || P.coarsest_is_correction);
            if ((int)g.M <= nthr) {
                tail_sweeps_cached<T, ND>(g, LL(last), CC(last), XA(last), XB(last), B(last), zero, 64, nthr);
            } else {
            tail_sweep<T, ND>(g, LL(last), CC(last), XA(last), B(last), XB(last), zero, nthr);
            for (int s = 1; s < 64; s += 2) {
                tail_sweep<T, ND>(g, LL(last), CC(last), XB(last), B(last), XA(last), false, nthr);
                if (s + 1 < 64) tail_sweep<T, ND>(g, LL(last), CC(last), XA(last), B(last), XB(last), false, nthr);
            }
            }
        }
    }
    // ---- up: x_l (in XA) += P x_{l+1} (in XA), 2 sweeps -> XA --------------------------------------------------------
    for (int l = last - 1; l >= 0; --l) {
        const Grid gf = P.g[l], gc = P.g[l + 1];
        const int nthr = nthr_of(l);
        // the threads of this level were idle while the coarser levels ran: wait for them with a barrier the coarser
        // level's threads also reach (all of them are threads of this level too)
        if ((int)threadIdx.x < nthr) {
            bar_sync_n(2 + l, nthr);   // one barrier id per level: several levels' idle threads wait at the same time
            T* x = XA(l);
            const T* xc = XA(l + 1);
            for (int I = threadIdx.x; I < (int)gf.M; I += nthr) {
                int i0, i1, i2;
                decompose_i<ND>(gf, I, i0, i1, i2);
                x[I] += xc[(i0 >> 1) + gc.N0 * ((i1 >> 1) + gc.N1 * (i2 >> 1))];
            }
            bar_sync_n(1, nthr);
            tail_sweep<T, ND>(gf, LL(l), CC(l), XA(l), B(l), XB(l), false, nthr);
            tail_sweep<T, ND>(gf, LL(l), CC(l), XB(l), B(l), XA(l), false, nthr);
        }
    }
    __syncthreads();
    {
        const int M = (int)P.g[0].M;
        const T* x0 = XA(0);
        for (int i = threadIdx.x; i < M; i += blockDim.x) P.x_out[i] = x0[i];
    }
}

}  // namespace wl
