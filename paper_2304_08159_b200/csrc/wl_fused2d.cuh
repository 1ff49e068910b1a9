// wl_fused2d.cuh — the level halves of the V-cycle as ONE kernel each, 2-D grids.
//
//   DOWN (H3+H4):  x2 = J(J(x0)),  bc = R (b - A x2)                     x0 = x_in [- mean] | 0
//   UP   (H6[+H7]): x2 = J(J(x0)),  x0 = x_in + P xc                      [+ ||b - A x2||inf and sum(x2) at level 0]
//
// A CTA owns a TX x TY tile.  The tile plus a halo of 3 (x: 4, whole 16-byte vectors) of x0, b, L0, L1 (and the coarse
// xc under it) arrives by TMA (2-D boxes, zero fill beyond the walls = Neumann), the three stencil stages run on
// shrinking rings with one __syncthreads between them, x1 and x2 live in shared memory only; a thread owns VEC
// consecutive cells (16 bytes) of a row and walks rows with stride RP.  2-D levels are small (BASELINE config 1:
// 4 MiB per array, L2-resident), so the kernel is latency-, not bandwidth-bound: one tile per CTA, several CTAs per SM.
// Expression order = the oracle's (upper face, lower face; axis 0, then 1; D summed per axis; IEEE division).
#pragma once
#include "wl_common.cuh"
#include "wl_fused3d.cuh"
#include "wl_tma.cuh"

namespace wl {

template <typename T, int TX_, int TY_>
struct F2 {
    static constexpr int VEC = 16 / (int)sizeof(T);
    static constexpr int TX = TX_, TY = TY_;
    static constexpr int HX = 4, HY = 3;
    static constexpr int WX = TX + 2 * HX, WY = TY + 2 * HY;
    static constexpr int NTX = WX / VEC;
    static constexpr int NT = 384;
    static constexpr int RP = NT / NTX;                          // rows per pass
    static constexpr int PLANE = WX * WY;
    static constexpr int PLANE_B = (PLANE * (int)sizeof(T) + 127) / 128 * 128;
    static constexpr int CH = (HX / 2 + VEC - 1) / VEC * VEC;    // coarse box starts on a 16-byte boundary (wl_fused3d.cuh)
    static constexpr int CWX = ((CH - HX / 2) + WX / 2 + VEC - 1) / VEC * VEC;
    static constexpr int CWY = WY / 2 + 1;
    static constexpr int CPLANE_B = (CWX * CWY * (int)sizeof(T) + 127) / 128 * 128;
    static constexpr int TX0 = HX / VEC, TX1 = NTX - HX / VEC;
    static_assert(TY / 2 <= RP, "one thread row per coarse row in the residual stage");
    static_assert(WX % VEC == 0 && TX % 2 == 0 && TY % 2 == 0, "tile geometry");
};

template <typename T>
struct Fused2Params {
    int N0, N1;
    int tiles_x, tiles_y;
    T* xout;
    T* bc;
    Scalars* scal;
    double* partials;
    double* hist;            // [TICKET] solve bookkeeping, as in Fused3Params
    Scalars* host_scal;
    double* host_hist;
    long long cells;
    int check_done;
};

// A x and D at the thread's VEC cells of row `me` of the shared plane xs (coefficients from the shared planes l0, l1).
template <typename T, int VEC, int WX>
__device__ __forceinline__ void apply_A2(const T* __restrict__ l0, const T* __restrict__ l1, const T* __restrict__ xs, int me,
                                         T (&xc)[VEC], T (&Ax)[VEC], T (&D)[VEC]) {
    T L0[VEC], L1[VEC], L1p[VEC], xS[VEC], xN[VEC];
    ld_vec<T, VEC>(l0 + me, L0);
    const T L0n = l0[me + VEC];
    ld_vec<T, VEC>(l1 + me, L1);
    ld_vec<T, VEC>(l1 + me + WX, L1p);
    ld_vec<T, VEC>(xs + me, xc);
    const T xW = xs[me - 1], xE = xs[me + VEC];
    ld_vec<T, VEC>(xs + me - WX, xS);
    ld_vec<T, VEC>(xs + me + WX, xN);
#pragma unroll
    for (int v = 0; v < VEC; ++v) {
        const T x = xc[v];
        const T Lxp = (v + 1 < VEC) ? L0[(v + 1) % VEC] : L0n;
        const T xe = (v + 1 < VEC) ? xc[(v + 1) % VEC] : xE;
        const T xw = (v > 0) ? xc[(v + VEC - 1) % VEC] : xW;
        T s = Lxp * (xe - x);
        s += L0[v] * (xw - x);
        s += L1p[v] * (xN[v] - x);
        s += L1[v] * (xS[v] - x);
        Ax[v] = s;
        D[v] = (L0[v] + Lxp) + (L1[v] + L1p[v]);
    }
}

template <typename T, int TX, int TY, bool PROLONG, bool ZERO_IN, bool SHIFT, bool STAGE3, bool RESTRICT, bool NORMS, bool RIN, bool TICKET>
__global__ void __launch_bounds__(F2<T, TX, TY>::NT)
k_fused2d(const __grid_constant__ CUtensorMap tm_x, const __grid_constant__ CUtensorMap tm_b,
          const __grid_constant__ CUtensorMap tm_L0, const __grid_constant__ CUtensorMap tm_L1,
          const __grid_constant__ CUtensorMap tm_xc, Fused2Params<T> P) {
    using G = F2<T, TX, TY>;
    constexpr int VEC = G::VEC, WX = G::WX, WY = G::WY, RP = G::RP;
    constexpr uint32_t TX_BYTES = (uint32_t)((ZERO_IN ? 3 : 4) * G::PLANE * sizeof(T) + (PROLONG ? G::CWX * G::CWY * sizeof(T) : 0));
    static_assert(!RESTRICT || STAGE3, "restriction comes out of the residual stage");
    static_assert(!(RIN && ZERO_IN), "a zero input has residual b");
    pdl_launch_dependents();   // the next kernel of the cycle may set up while this one runs (it waits before touching data)

    extern __shared__ __align__(1024) unsigned char smem2[];
    uint64_t* bar = (uint64_t*)smem2;
    auto arr = [&](int a) -> T* { return (T*)(smem2 + 128 + a * G::PLANE_B); };   // 0 x0, 1 b, 2 L0, 3 L1, 4 x1, 5 x2, 6 xc
    T* sx0 = arr(0); T* sb = arr(1); T* sl0 = arr(2); T* sl1 = arr(3); T* sx1 = arr(4); T* sx2 = arr(5); T* sxc = arr(6);

    const int t = threadIdx.x;
    const int ty0 = t / G::NTX, tx = t - ty0 * G::NTX;
    const bool active = ty0 < RP;
    const int tile = blockIdx.x;
    const int tyi = tile / P.tiles_x, txi = tile - tyi * P.tiles_x;
    const int X0 = txi * TX, Y0 = tyi * TY;
    const T omega = Omega<T>::value();

    if (t == 0) {
        mbar_init(bar, 1);        // coefficients
        mbar_init(bar + 1, 1);    // x, b, xc
        fence_mbar_init();
    }
    __syncthreads();
    // The coefficients are written by no kernel of a cycle (and a kernel launched with the programmatic attribute always
    // follows another kernel of the same cycle): their tiles are fetched while the predecessor is still draining.
    if (t == 0) {
        mbar_expect_tx(bar, (uint32_t)(2 * G::PLANE * sizeof(T)));
        tma_load_2d(sl0, &tm_L0, X0 - G::HX, Y0 - G::HY, bar);
        tma_load_2d(sl1, &tm_L1, X0 - G::HX, Y0 - G::HY, bar);
    }
    pdl_wait();
    if (P.check_done && P.scal->done) {   // uniform; no CTA may exit with a bulk copy into its shared memory in flight
        mbar_wait(bar, 0);
        return;
    }
    if (t == 0) {
        mbar_expect_tx(bar + 1, TX_BYTES - (uint32_t)(2 * G::PLANE * sizeof(T)));
        if constexpr (!ZERO_IN) tma_load_2d(sx0, &tm_x, X0 - G::HX, Y0 - G::HY, bar + 1);
        tma_load_2d(sb, &tm_b, X0 - G::HX, Y0 - G::HY, bar + 1);
        if constexpr (PROLONG) tma_load_2d(sxc, &tm_xc, X0 / 2 - G::CH, Y0 / 2 - 2, bar + 1);
    }
    mbar_wait(bar, 0);
    mbar_wait(bar + 1, 0);

    // ---- stage 0: x0 += P xc, x0 -= mean (in place) -------------------------------------------------------------------
    if constexpr (!ZERO_IN && (PROLONG || SHIFT)) {
        T shift = (T)0;
        if constexpr (SHIFT) shift = (T)P.scal->shift;
        if (active)
            for (int ty = ty0; ty < WY; ty += RP) {
                const int me = ty * WX + tx * VEC;
                T v[VEC];
                ld_vec<T, VEC>(sx0 + me, v);
#pragma unroll
                for (int k = 0; k < VEC; ++k) {
                    if constexpr (PROLONG) v[k] += sxc[((ty + 1) >> 1) * G::CWX + (G::CH - G::HX / 2) + tx * (VEC / 2) + (k >> 1)];
                    if constexpr (SHIFT) v[k] -= shift;
                }
                st_vec<T, VEC>(sx0 + me, v);
            }
        __syncthreads();
    }
    T rmax = (T)0;
    // ---- stage 1: x1 on rows 1 .. WY-2 ---------------------------------------------------------------------------------
    if (active)
        for (int ty = 1 + ty0; ty <= WY - 2; ty += RP) {
            const int me = ty * WX + tx * VEC;
            T xc[VEC], Ax[VEC], D[VEC], bb[VEC], x1[VEC];
            ld_vec<T, VEC>(sb + me, bb);
            if constexpr (ZERO_IN) {
                T L0[VEC], L1[VEC], L1p[VEC];
                ld_vec<T, VEC>(sl0 + me, L0);
                const T L0n = sl0[me + VEC];
                ld_vec<T, VEC>(sl1 + me, L1);
                ld_vec<T, VEC>(sl1 + me + WX, L1p);
#pragma unroll
                for (int v = 0; v < VEC; ++v) {
                    const T Lxp = (v + 1 < VEC) ? L0[(v + 1) % VEC] : L0n;
                    const T Dv = (L0[v] + Lxp) + (L1[v] + L1p[v]);
                    const T c = (Dv > (T)0) ? omega * ((T)1 / Dv) : (T)0;
                    x1[v] = c * ((T)0 - bb[v]);
                }
            } else {
                apply_A2<T, VEC, WX>(sl0, sl1, sx0, me, xc, Ax, D);
                const int gx = X0 - G::HX + tx * VEC, gy = Y0 - G::HY + ty;
                const bool inside = tx >= G::TX0 && tx < G::TX1 && ty >= G::HY && ty < WY - G::HY && gx < P.N0 && gy < P.N1;
#pragma unroll
                for (int v = 0; v < VEC; ++v) {
                    const T c = (D[v] > (T)0) ? omega * ((T)1 / D[v]) : (T)0;
                    const T d = Ax[v] - bb[v];
                    if constexpr (RIN) {
                        if (inside) rmax = (d != d || rmax != rmax) ? (rmax + d) : fmax(rmax, fabs(d));
                    }
                    x1[v] = xc[v] + c * d;
                }
            }
            st_vec<T, VEC>(sx1 + me, x1);
        }
    __syncthreads();
    // ---- stage 2: x2 on rows 2 .. WY-3; interior cells go to HBM ---------------------------------------------------------
    double psum = 0.0;
    if (active)
        for (int ty = 2 + ty0; ty <= WY - 3; ty += RP) {
            const int me = ty * WX + tx * VEC;
            T xc[VEC], Ax[VEC], D[VEC], bb[VEC], x2[VEC];
            ld_vec<T, VEC>(sb + me, bb);
            apply_A2<T, VEC, WX>(sl0, sl1, sx1, me, xc, Ax, D);
#pragma unroll
            for (int v = 0; v < VEC; ++v) {
                const T c = (D[v] > (T)0) ? omega * ((T)1 / D[v]) : (T)0;
                x2[v] = xc[v] + c * (Ax[v] - bb[v]);
            }
            st_vec<T, VEC>(sx2 + me, x2);
            const int gx = X0 - G::HX + tx * VEC, gy = Y0 - G::HY + ty;
            if (tx >= G::TX0 && tx < G::TX1 && ty >= G::HY && ty < WY - G::HY && gx < P.N0 && gy < P.N1) {
                st_vec<T, VEC>(P.xout + (size_t)gy * P.N0 + gx, x2);
                if constexpr (NORMS) {
#pragma unroll
                    for (int v = 0; v < VEC; ++v) psum += (double)x2[v];
                }
            }
        }
    // ---- stage 3: r = b - A x2 on the tile; one thread row per coarse row ------------------------------------------------
    if constexpr (STAGE3) {
        __syncthreads();
        if (active && ty0 < TY / 2 && tx >= G::TX0 && tx < G::TX1) {
            T rs[VEC / 2 > 0 ? VEC / 2 : 1];
#pragma unroll
            for (int k = 0; k < VEC / 2; ++k) rs[k] = (T)0;
            T rowsum[2][VEC / 2 > 0 ? VEC / 2 : 1];
            const int gx = X0 - G::HX + tx * VEC;
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int ty = G::HY + 2 * ty0 + h;
                const int me = ty * WX + tx * VEC;
                const int gy = Y0 - G::HY + ty;
                T xc[VEC], Ax[VEC], D[VEC], bb[VEC], r[VEC];
                ld_vec<T, VEC>(sb + me, bb);
                apply_A2<T, VEC, WX>(sl0, sl1, sx2, me, xc, Ax, D);
#pragma unroll
                for (int v = 0; v < VEC; ++v) r[v] = bb[v] - Ax[v];
#pragma unroll
                for (int v = 0; v < VEC; v += 2) rowsum[h][v >> 1] = r[v] + r[v + 1];
                if constexpr (NORMS && !RIN) {
                    if (gx < P.N0 && gy < P.N1) {
#pragma unroll
                        for (int v = 0; v < VEC; ++v) rmax = (r[v] != r[v] || rmax != rmax) ? (rmax + r[v]) : fmax(rmax, fabs(r[v]));
                    }
                }
            }
            if constexpr (RESTRICT) {
                const int C0 = P.N0 >> 1, C1 = P.N1 >> 1;
                const int gcy = (Y0 >> 1) + ty0;
                const int gcx = (gx >> 1);
                if (gcy < C1) {
#pragma unroll
                    for (int k = 0; k < VEC / 2; ++k)
                        if (gcx + k < C0) P.bc[(size_t)gcy * C0 + gcx + k] = rowsum[0][k] + rowsum[1][k];
                }
            }
            (void)rs;
        }
    }
    if constexpr (NORMS || RIN) {
        __shared__ double red[32];
        if constexpr ((NORMS && STAGE3) || RIN) {
            const double m = block_max((double)rmax, red);
            if (t == 0) atomic_max_nonneg(&P.scal->absmax_bits[1], m);
        }
        if constexpr (NORMS) {
            const double s = block_sum(psum, red);
            if (t == 0) P.partials[blockIdx.x] = s;
        }
        if constexpr (TICKET) {   // the last CTA to finish does the cycle's bookkeeping (wl_fused3d.cuh)
            __shared__ int s_last;
            if (t == 0) {
                __threadfence();
                const unsigned int ticket = atomicAdd(&P.scal->ticket, 1u);
                s_last = (ticket == gridDim.x - 1) ? 1 : 0;
            }
            __syncthreads();
            if (s_last && t < 32) {
                __threadfence();
                if constexpr (RIN) {
                    if (t == 0) solve_check_lagged(P.scal, P.hist, P.host_scal, P.host_hist);
                } else {
                    solve_finish_mean_lagged(P.scal, P.partials, (int)gridDim.x, P.cells);
                }
                if (t == 0) P.scal->ticket = 0u;
            }
        }
    }
}

template <typename T, int TX, int TY>
constexpr size_t fused2d_smem_bytes() {
    using G = F2<T, TX, TY>;
    return 128 + 6 * (size_t)G::PLANE_B + G::CPLANE_B;
}

}  // namespace wl
