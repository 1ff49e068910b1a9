// wl_tail.cuh — the coarse tail of the V-cycle in ONE persistent CTA (H5; BJ "Small coarse levels in a single persistent
// CTA"): every level from `first` down to the coarsest lives in shared memory (x ping-pong, b, L); the CTA walks
// down (2 sweeps, residual, restriction), does the 64 coarsest sweeps, and walks up (injection, 2 sweeps) with
// __syncthreads between steps — no launches, no HBM traffic beyond reading b, L once and writing x once.
// The arithmetic per cell is the generic kernels' (stencil_cell), i.e. the oracle's expression order.
#pragma once
#include "wl_common.cuh"
#include "wl_generic.cuh"

namespace wl {

constexpr int kTailMaxLevels = 8;
constexpr int kTailThreads = 1024;

template <typename T>
struct TailParams {
    int nl;                          // levels in the tail (>= 1); level 0 of the tail = `first` of the hierarchy
    int zero_in;                     // 1: start from x = 0 on the tail's first level; 0: start from x_in
    Grid g[kTailMaxLevels];
    const T* L[kTailMaxLevels];      // global coefficient arrays of each tail level
    unsigned off[kTailMaxLevels];    // byte offset of the level's block in shared memory: xA, xB, b, L (ND arrays)
    const T* x_in;                   // tail level 0 initial guess (ignored if zero_in)
    const T* b_in;                   // tail level 0 right-hand side (global)
    T* x_out;                        // tail level 0 result (global)
    int coarsest_is_correction;      // 1: the coarsest level starts from 0 (it is a correction level of the hierarchy)
};

template <typename T, int ND>
__device__ __forceinline__ void tail_sweep(const Grid& g, const T* L, const T* xin, const T* b, T* xout, bool from_zero) {
    const T omega = Omega<T>::value();
    for (int I = threadIdx.x; I < (int)g.M; I += blockDim.x) {
        int i0, i1, i2;
        decompose<T, ND>(g, I, i0, i1, i2);
        if (from_zero) {
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
            xout[I] = omega * invD * ((T)0 - b[I]);
        } else {
            T Ax, D;
            stencil_cell<T, ND>(g, L, xin, I, i0, i1, i2, Ax, D);
            const T invD = (D > (T)0) ? (T)1 / D : (T)0;
            xout[I] = xin[I] + omega * invD * (Ax - b[I]);
        }
    }
    __syncthreads();
}

template <typename T, int ND>
__global__ void __launch_bounds__(kTailThreads, 1) k_coarse_tail(TailParams<T> P) {
    extern __shared__ __align__(16) unsigned char tail_smem[];
    auto XA = [&](int l) -> T* { return (T*)(tail_smem + P.off[l]); };
    auto XB = [&](int l) -> T* { return XA(l) + P.g[l].M; };
    auto B = [&](int l) -> T* { return XA(l) + 2 * P.g[l].M; };
    auto LL = [&](int l) -> T* { return XA(l) + 3 * P.g[l].M; };

    // stage every level's coefficients, and the first level's b (and x) in shared memory
    for (int l = 0; l < P.nl; ++l) {
        const int n = (int)P.g[l].M * ND;
        T* d = LL(l);
        for (int i = threadIdx.x; i < n; i += blockDim.x) d[i] = P.L[l][i];
    }
    {
        const int M = (int)P.g[0].M;
        T* b0 = B(0);
        T* x0 = XA(0);
        for (int i = threadIdx.x; i < M; i += blockDim.x) {
            b0[i] = P.b_in[i];
            if (!P.zero_in) x0[i] = P.x_in[i];
        }
    }
    __syncthreads();

    const int last = P.nl - 1;
    // ---- down ----------------------------------------------------------------------------------------------------
    for (int l = 0; l < last; ++l) {
        const Grid gf = P.g[l], gc = P.g[l + 1];
        const bool zero = (l > 0) || P.zero_in;
        tail_sweep<T, ND>(gf, LL(l), XA(l), B(l), XB(l), zero);      // XA -> XB
        tail_sweep<T, ND>(gf, LL(l), XB(l), B(l), XA(l), false);     // XB -> XA  (x after 2 pre-sweeps)
        const T* x = XA(l);
        const T* b = B(l);
        const T* L = LL(l);
        T* bc = B(l + 1);
        for (int J = threadIdx.x; J < (int)gc.M; J += blockDim.x) {  // b_{l+1} = R (b - A x): pairwise along 0, 1, 2
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
        }
        __syncthreads();
    }
    // ---- coarsest: 64 sweeps, result in XA(last) ---------------------------------------------------------------------
    {
        const Grid g = P.g[last];
        const bool zero = (last > 0) ? true : (P.zero_in || P.coarsest_is_correction);
        tail_sweep<T, ND>(g, LL(last), XA(last), B(last), XB(last), zero);
        for (int s = 1; s < 64; s += 2) {
            tail_sweep<T, ND>(g, LL(last), XB(last), B(last), XA(last), false);
            if (s + 1 < 64) tail_sweep<T, ND>(g, LL(last), XA(last), B(last), XB(last), false);
        }
    }
    // ---- up: x_l (in XA) += P x_{l+1} (in XA), 2 sweeps -> XA --------------------------------------------------------
    for (int l = last - 1; l >= 0; --l) {
        const Grid gf = P.g[l], gc = P.g[l + 1];
        T* x = XA(l);
        const T* xc = XA(l + 1);
        for (int I = threadIdx.x; I < (int)gf.M; I += blockDim.x) {
            int i0, i1, i2;
            decompose<T, ND>(gf, I, i0, i1, i2);
            x[I] += xc[cell_index(gc, i0 >> 1, i1 >> 1, i2 >> 1)];
        }
        __syncthreads();
        tail_sweep<T, ND>(gf, LL(l), XA(l), B(l), XB(l), false);
        tail_sweep<T, ND>(gf, LL(l), XB(l), B(l), XA(l), false);
    }
    {
        const int M = (int)P.g[0].M;
        const T* x0 = XA(0);
        for (int i = threadIdx.x; i < M; i += blockDim.x) P.x_out[i] = x0[i];
    }
}

}  // namespace wl
