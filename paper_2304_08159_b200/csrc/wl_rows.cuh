// wl_rows.cuh — the streaming steps of the projection (H0 level-0 copy, H1 divergence, H8 gradient correction) as
// row-wise kernels with 16-byte loads and stores along the unit-stride axis (BJ "vectorised 16-byte coalesced loads
// along the unit-stride axis", "Fused divergence and pressure-gradient kernels over all n directions").
// A CTA is (32·k) x-lanes by RY rows; a (component,) z, y row index costs two integer divisions per ROW, none per cell.
// Same expressions, same order as the generic kernels (and the oracle): results are bit-identical to them.
// Used when N_0 is a multiple of the vector width and the arrays are 16-byte aligned; otherwise the generic kernels run.
#pragma once
#include "wl_common.cuh"
#include "wl_fused3d.cuh"  // ld_vec / st_vec
#include "wl_generic.cuh"  // decompose

namespace wl {

constexpr int kRowsX = 64, kRowsY = 4;   // CTA shape: 64 vector lanes x 4 rows

// H0, level 0: Lout = Lin with the wall plane I_i = 0 of component i forced to 0.
template <typename T, int ND>
__global__ void __launch_bounds__(kRowsX* kRowsY) k_copy_coeff_rows(Grid g, const T* __restrict__ Lin, T* __restrict__ Lout) {
    constexpr int VEC = 16 / (int)sizeof(T);
    const int nvx = g.N0 / VEC;
    const long long rows_per_comp = (long long)g.N1 * g.N2;
    const long long nrows = rows_per_comp * ND;
    for (long long r = (long long)blockIdx.x * kRowsY + threadIdx.y; r < nrows; r += (long long)gridDim.x * kRowsY) {
        const int comp = (int)(r / rows_per_comp);
        const long long rc = r - (long long)comp * rows_per_comp;
        const int z = (int)(rc / g.N1), y = (int)(rc - (long long)z * g.N1);
        const bool wall_row = (comp == 1 && y == 0) || (comp == 2 && z == 0);
        const T* src = Lin + r * g.N0;
        T* dst = Lout + r * g.N0;
        for (int vx = threadIdx.x; vx < nvx; vx += kRowsX) {
            T v[VEC];
            ld_vec<T, VEC>(src + vx * VEC, v);
            if (wall_row) {
#pragma unroll
                for (int k = 0; k < VEC; ++k) v[k] = (T)0;
            } else if (comp == 0 && vx == 0) {
                v[0] = (T)0;
            }
            st_vec<T, VEC>(dst + vx * VEC, v);
        }
    }
}

// H1: b[I] = sum_i (u[i][I+d_i] - u[i][I]), unstored upper wall face = 0.
template <typename T, int ND>
__global__ void __launch_bounds__(kRowsX* kRowsY) k_divergence_rows(Grid g, const T* __restrict__ u, T* __restrict__ b,
                                                                   Scalars* scal /* nullable: ||b||inf -> slot 0 */) {
    constexpr int VEC = 16 / (int)sizeof(T);
    const int nvx = g.N0 / VEC;
    const long long nrows = (long long)g.N1 * g.N2;
    const long long sy = g.N0, sz = (long long)g.N0 * g.N1;
    T bmax = (T)0;
    for (long long r = (long long)blockIdx.x * kRowsY + threadIdx.y; r < nrows; r += (long long)gridDim.x * kRowsY) {
        const int z = (int)(r / g.N1), y = (int)(r - (long long)z * g.N1);
        const T* u0 = u + r * g.N0;
        const T* u1 = u0 + g.M;
        const T* u2 = u1 + g.M;
        const bool up1 = (y + 1 < g.N1), up2 = (ND == 3) && (z + 1 < g.N2);
        for (int vx = threadIdx.x; vx < nvx; vx += kRowsX) {
            const int x = vx * VEC;
            T a0[VEC], a1[VEC], a1p[VEC], out[VEC];
            ld_vec<T, VEC>(u0 + x, a0);
            const T a0n = (x + VEC < g.N0) ? u0[x + VEC] : (T)0;
            ld_vec<T, VEC>(u1 + x, a1);
            if (up1) ld_vec<T, VEC>(u1 + x + sy, a1p);
            else {
#pragma unroll
                for (int k = 0; k < VEC; ++k) a1p[k] = (T)0;
            }
            T a2[VEC], a2p[VEC];
            if (ND == 3) {
                ld_vec<T, VEC>(u2 + x, a2);
                if (up2) ld_vec<T, VEC>(u2 + x + sz, a2p);
                else {
#pragma unroll
                    for (int k = 0; k < VEC; ++k) a2p[k] = (T)0;
                }
            }
#pragma unroll
            for (int k = 0; k < VEC; ++k) {
                const T e = (k + 1 < VEC) ? a0[(k + 1) % VEC] : a0n;
                T s = 0;
                s += e - a0[k];
                s += a1p[k] - a1[k];
                if (ND == 3) s += a2p[k] - a2[k];
                out[k] = s;
                bmax = (s != s || bmax != bmax) ? (bmax + s) : fmax(bmax, fabs(s));
            }
            st_vec<T, VEC>(b + r * g.N0 + x, out);
        }
    }
    if (scal) {   // uniform branch: every thread of the CTA takes it
        __shared__ double red[32];
        double m = warp_max((double)bmax);
        const int tid = threadIdx.y * kRowsX + threadIdx.x;
        if ((tid & 31) == 0) red[tid >> 5] = m;
        __syncthreads();
        if (tid < 32) {
            m = (tid < (kRowsX * kRowsY) / 32) ? red[tid] : 0.0;
            m = warp_max(m);
            if (tid == 0) atomic_max_nonneg(&scal->absmax_bits[0], m);
        }
    }
}

// H8: u[i][I] -= L[i][I] (p[I] - p[I-d_i]) for all i; wall planes I_i = 0 untouched.
template <typename T, int ND>
__global__ void __launch_bounds__(kRowsX* kRowsY) k_gradient_rows(Grid g, const T* __restrict__ L, T* __restrict__ u,
                                                                 const T* __restrict__ p) {
    constexpr int VEC = 16 / (int)sizeof(T);
    const int nvx = g.N0 / VEC;
    const long long nrows = (long long)g.N1 * g.N2;
    const long long sy = g.N0, sz = (long long)g.N0 * g.N1;
    for (long long r = (long long)blockIdx.x * kRowsY + threadIdx.y; r < nrows; r += (long long)gridDim.x * kRowsY) {
        const int z = (int)(r / g.N1), y = (int)(r - (long long)z * g.N1);
        const T* pr = p + r * g.N0;
        for (int vx = threadIdx.x; vx < nvx; vx += kRowsX) {
            const int x = vx * VEC;
            const long long e0 = r * g.N0 + x;
            T pc[VEC];
            ld_vec<T, VEC>(pr + x, pc);
            {   // direction 0
                const T pw = (x > 0) ? pr[x - 1] : (T)0;
                T l[VEC], uu[VEC];
                ld_vec<T, VEC>(L + e0, l);
                ld_vec<T, VEC>(u + e0, uu);
#pragma unroll
                for (int k = 0; k < VEC; ++k) {
                    const T pm = (k > 0) ? pc[(k + VEC - 1) % VEC] : pw;
                    if (x + k > 0) uu[k] -= l[k] * (pc[k] - pm);
                }
                st_vec<T, VEC>(u + e0, uu);
            }
            if (y > 0) {   // direction 1
                T pm[VEC], l[VEC], uu[VEC];
                ld_vec<T, VEC>(pr + x - sy, pm);
                ld_vec<T, VEC>(L + g.M + e0, l);
                ld_vec<T, VEC>(u + g.M + e0, uu);
#pragma unroll
                for (int k = 0; k < VEC; ++k) uu[k] -= l[k] * (pc[k] - pm[k]);
                st_vec<T, VEC>(u + g.M + e0, uu);
            }
            if (ND == 3 && z > 0) {   // direction 2
                T pm[VEC], l[VEC], uu[VEC];
                ld_vec<T, VEC>(pr + x - sz, pm);
                ld_vec<T, VEC>(L + 2 * g.M + e0, l);
                ld_vec<T, VEC>(u + 2 * g.M + e0, uu);
#pragma unroll
                for (int k = 0; k < VEC; ++k) uu[k] -= l[k] * (pc[k] - pm[k]);
                st_vec<T, VEC>(u + 2 * g.M + e0, uu);
            }
        }
    }
}

// C = omega * invD per cell, D = sum of the cell's 2n face coefficients in the oracle's order ((Lm + Lp) per axis, axes
// 0, 1, 2), invD = D > 0 ? 1/D : 0 with IEEE division: exactly the factor the oracle forms in every sweep.  Computed
// once per coefficient set and level; the fused kernels load it instead of recomputing D and a reciprocal per sweep.
template <typename T, int ND>
__global__ void __launch_bounds__(kRowsX* kRowsY) k_make_c_rows(Grid g, const T* __restrict__ L, T* __restrict__ C) {
    constexpr int VEC = 16 / (int)sizeof(T);
    const int nvx = g.N0 / VEC;
    const long long nrows = (long long)g.N1 * g.N2;
    const long long sy = g.N0, sz = (long long)g.N0 * g.N1;
    const T omega = Omega<T>::value();
    for (long long r = (long long)blockIdx.x * kRowsY + threadIdx.y; r < nrows; r += (long long)gridDim.x * kRowsY) {
        const int z = (int)(r / g.N1), y = (int)(r - (long long)z * g.N1);
        const T* l0 = L + r * g.N0;
        const T* l1 = l0 + g.M;
        const T* l2 = l1 + g.M;
        const bool up1 = (y + 1 < g.N1), up2 = (ND == 3) && (z + 1 < g.N2);
        for (int vx = threadIdx.x; vx < nvx; vx += kRowsX) {
            const int x = vx * VEC;
            T a0[VEC], a1[VEC], a1p[VEC], a2[VEC], a2p[VEC], out[VEC];
            ld_vec<T, VEC>(l0 + x, a0);
            const T a0n = (x + VEC < g.N0) ? l0[x + VEC] : (T)0;
            ld_vec<T, VEC>(l1 + x, a1);
            if (up1) ld_vec<T, VEC>(l1 + x + sy, a1p);
            if (ND == 3) {
                ld_vec<T, VEC>(l2 + x, a2);
                if (up2) ld_vec<T, VEC>(l2 + x + sz, a2p);
            }
#pragma unroll
            for (int k = 0; k < VEC; ++k) {
                const T e = (k + 1 < VEC) ? a0[(k + 1) % VEC] : a0n;
                // wall faces: the stored plane I_i = 0 is already 0 in the library's copy; the unstored upper wall is 0
                T D = 0;
                D += a0[k] + e;
                D += a1[k] + (up1 ? a1p[k] : (T)0);
                if (ND == 3) D += a2[k] + (up2 ? a2p[k] : (T)0);
                const T invD = (D > (T)0) ? (T)1 / D : (T)0;
                out[k] = omega * invD;
            }
            st_vec<T, VEC>(C + r * g.N0 + x, out);
        }
    }
}
// Any-shape version (rows that are not whole vectors).
template <typename T, int ND>
__global__ void k_make_c(Grid g, const T* __restrict__ L, T* __restrict__ C) {
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
        C[I] = omega * invD;
    }
}

}  // namespace wl
