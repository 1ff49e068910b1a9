// wl_convdiff.cuh — NEXT-4: the convection + diffusion rate of change of the face velocity, the paper's
// `convdiff!` routine ("a third-order finite volume scheme ... implicit Large Eddy Simulation",
// PAPER.md:25).  The text names the scheme only; every detail is DESIGN.md §3 reading 15:
//   r[i][I] = sum_j ( F_ij(I) - F_ij(I + d_j) )  on faces I_i >= 1,  r = 0 on the stored wall plane I_i = 0,
//   F_ij(I) = U phi - nu (u[i][I] - u[i][I - d_j]),   U = (u[j][I] + u[j][I - d_i]) / 2,
//   phi     = median(phi3, C, median(C, D, 10 C - 9 UU)),  phi3 = (5 C + 2 D - UU) / 6,  with C / D the values of u_i up /
//             downstream of the flux point and UU the one beyond C (U >= 0: C = u[i][I-d_j], D = u[i][I], UU = u[i][I-2d_j];
//             U < 0: C = u[i][I], D = u[i][I-d_j], UU = u[i][I+d_j]);  phi = (C + D) / 2 where UU lies outside the field;
//   closed free-slip box: F_ij = 0 on the walls I_j = 0, N_j for j != i; the unstored upper wall value u[i][N_i] is 0.
// Every operation rounds separately and in the order written (the library is compiled with -fmad=false); the medians are taken
// with min / max, which pick the same VALUE as any comparison network (the sign of a zero may differ; NaN inputs are out of
// contract), so for finite fields r equals the oracle's value for value.
//
// Two kernels: k_convdiff (any shape, 2-D / 3-D, one thread per cell, every flux evaluated by both cells it separates) and
// k_convdiff3d (3-D, rows of whole 16-byte vectors): a CTA owns a 32·VEC x TY tile and marches along z; planes arrive by TMA
// into a six-slot ring (zero fill beyond the box = the unstored upper wall values; planes k-2 .. k+1 are read from the ring, two
// more are in flight); a warp is one row, a thread owns one 16-byte vector of it; every flux is evaluated ONCE (x: 4+1 per
// thread; y: handed to the row below through shared memory, one more warp evaluates the row above the tile; z: the lower-face
// flux of plane k completes plane k-1 and is parked in shared memory for the next step).  DESIGN.md §6.6 has the measurements.
#pragma once
#include <cuda.h>

#include <type_traits>

#include "wl_common.cuh"
#include "wl_fused3d.cuh"
#include "wl_generic.cuh"
#include "wl_tma.cuh"

namespace wl {

__device__ __forceinline__ float cd_min(float a, float b) { return fminf(a, b); }
__device__ __forceinline__ float cd_max(float a, float b) { return fmaxf(a, b); }
__device__ __forceinline__ double cd_min(double a, double b) { return fmin(a, b); }
__device__ __forceinline__ double cd_max(double a, double b) { return fmax(a, b); }

template <typename T>
__device__ __forceinline__ T cd_med3(T a, T b, T c) {
    return cd_max(cd_min(a, b), cd_min(cd_max(a, b), c));
}
__device__ __forceinline__ float cd_min3(float a, float b, float c) {   // FMNMX3 (sm_100)
    float r;
    asm("min.f32 %0, %1, %2, %3;" : "=f"(r) : "f"(a), "f"(b), "f"(c));
    return r;
}
__device__ __forceinline__ double cd_min3(double a, double b, double c) { return fmin(fmin(a, b), c); }
// +1 or -1 with the sign of d (d = D - C): multiplying the limiter's arguments by it mirrors a falling profile into a rising one.
__device__ __forceinline__ float cd_sign1(float d) { return __uint_as_float((__float_as_uint(d) & 0x80000000u) | 0x3f800000u); }
__device__ __forceinline__ double cd_sign1(double d) {
    return __longlong_as_double((long long)(((unsigned long long)__double_as_longlong(d) & 0x8000000000000000ULL) | 0x3ff0000000000000ULL));
}
// median(phi3, C, median(C, D, bound)) for C <= D: the inner median is min(max(bound, C), D) >= C, so the outer one clamps
// phi3 to [C, inner] — three instructions, the last a three-input minimum.  Same value as the comparison network.
template <typename T>
__device__ __forceinline__ T cd_limit_rising(T phi3, T C, T D, T bound) {
    return cd_min3(cd_max(phi3, C), cd_max(bound, C), D);
}

// x / 6, correctly rounded.  fp32, fast form: q = RN(x·RN(1/6)), one exact remainder, one correction — equal to the IEEE
// quotient for every finite x with |x| >= 2^-100 (all mantissas checked on the host: tests/test_div6.py) and for x = 0 up to
// the sign of the zero.  Smaller non-zero magnitudes (a subnormal quotient) raise `tiny`, and the caller evaluates its group
// of fluxes again with the division proper (EXACT): the hot path carries two integer instructions per flux instead of a
// division sequence.
template <bool EXACT>
__device__ __forceinline__ float cd_div6(float x, bool& tiny) {
    if constexpr (EXACT) {
        return x / 6.0f;
    } else {
        const float y = 0.16666667163372039794921875f;   // RN(1/6)
        const float q = __fmul_rn(x, y);
        const float r = fmaf(-6.0f, q, x);
        // 0 < |x| < 2^-100 on the bit pattern (the sign shifted out, zero wrapped to the top): one multiply-add, one compare
        tiny = tiny || (__float_as_uint(x) * 2u - 2u < 2u * 0x0D800000u - 2u);
        return fmaf(r, y, q);
    }
}
template <bool EXACT>
__device__ __forceinline__ double cd_div6(double x, bool&) { return x / 6.0; }

// Boundary flags travel as bit masks (all ones = true): `have ? a : b` is then one bitwise select, and a flag that is a
// compile-time constant (the interior x-positions of a thread's vector) folds away.
template <typename T> struct CdMask;
template <> struct CdMask<float> { typedef unsigned int type; };
template <> struct CdMask<double> { typedef unsigned long long type; };
__device__ __forceinline__ float cd_bitsel(unsigned int m, float a, float b) {
    return __uint_as_float((__float_as_uint(a) & m) | (__float_as_uint(b) & ~m));
}
__device__ __forceinline__ double cd_bitsel(unsigned long long m, double a, double b) {
    return __longlong_as_double((long long)(((unsigned long long)__double_as_longlong(a) & m) | ((unsigned long long)__double_as_longlong(b) & ~m)));
}

// One face flux.  (a, b): the two values of the advecting component; m2, m1, p0, p1: the advected component at I-2d, I-d, I,
// I+d along the flux direction; hm2 / hp1: whether I-2d / I+d lie inside the field; wall: the face lies on an impermeable wall.
template <typename T, bool EXACT>
__device__ __forceinline__ T cd_flux(T a, T b, T m2, T m1, T p0, T p1, typename CdMask<T>::type hm2, typename CdMask<T>::type hp1,
                                     typename CdMask<T>::type wall, T nu, bool& tiny) {
    const T U = T(0.5) * (a + b);
    const bool pos = U >= T(0);
    const T C = pos ? m1 : p0;
    const T D = pos ? p0 : m1;
    const T UU = pos ? m2 : p1;
    const typename CdMask<T>::type have = pos ? hm2 : hp1;
    // mirrored so that D' >= C' (negation commutes with every rounding below, so phi = sg * phi' exactly)
    const T sg = cd_sign1(D - C);
    const T Cm = sg * C, Dm = sg * D, UUm = sg * UU;
    const T phi3 = cd_div6<EXACT>(T(5) * Cm + T(2) * Dm - UUm, tiny);
    const T bound = T(10) * Cm - T(9) * UUm;
    const T lim = cd_limit_rising(phi3, Cm, Dm, bound);
    const T cen = T(0.5) * (Cm + Dm);
    const T phi = sg * cd_bitsel(have, lim, cen);
    return cd_bitsel(wall, T(0), U * phi - nu * (p0 - m1));
}

// Two fluxes side by side (fp32): the additions and multiplications run as packed f32x2 instructions (two IEEE-rounded results
// per issue slot; a product is fma(a, b, -0), see wl_fused3d.cuh), selects, medians and the tiny test stay per element.
struct CdConst2 { u64 half, two, five, six_neg, nine, ten, y, nu, nz; };
template <bool EXACT>
__device__ __forceinline__ void cd_flux2(u64 a, u64 b, u64 m2, u64 m1, u64 p0, u64 p1, unsigned hm2, unsigned hp1, unsigned wall,
                                         const CdConst2& k, bool& tiny, float& f0, float& f1) {
    const u64 U = f2_mul(k.half, f2_add(a, b), k.nz);
    float U0, U1, m20, m21, m10, m11, p00, p01, p10, p11;
    f2_unpack(U, U0, U1);
    f2_unpack(m2, m20, m21); f2_unpack(m1, m10, m11); f2_unpack(p0, p00, p01); f2_unpack(p1, p10, p11);
    const bool pos0 = U0 >= 0.0f, pos1 = U1 >= 0.0f;
    const float C0 = pos0 ? m10 : p00, C1 = pos1 ? m11 : p01;
    const float D0 = pos0 ? p00 : m10, D1 = pos1 ? p01 : m11;
    const float UU0 = pos0 ? m20 : p10, UU1 = pos1 ? m21 : p11;
    const unsigned have0 = pos0 ? hm2 : hp1, have1 = pos1 ? hm2 : hp1;
    const u64 Cu = f2_pack(C0, C1), Du = f2_pack(D0, D1);
    float d0, d1;
    f2_unpack(f2_sub(Du, Cu), d0, d1);
    const u64 sg = f2_pack(cd_sign1(d0), cd_sign1(d1));   // mirror each flux so that D >= C (see cd_flux)
    const u64 C = f2_mul(sg, Cu, k.nz), D = f2_mul(sg, Du, k.nz), UU = f2_mul(sg, f2_pack(UU0, UU1), k.nz);
    const u64 x = f2_sub(f2_add(f2_mul(k.five, C, k.nz), f2_mul(k.two, D, k.nz)), UU);
    float phi30, phi31;
    if constexpr (EXACT) {
        float x0, x1;
        f2_unpack(x, x0, x1);
        phi30 = x0 / 6.0f;
        phi31 = x1 / 6.0f;
    } else {
        const u64 q = f2_mul(x, k.y, k.nz);
        u64 r, q2;
        asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(k.six_neg), "l"(q), "l"(x));
        asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(q2) : "l"(r), "l"(k.y), "l"(q));
        f2_unpack(q2, phi30, phi31);
        tiny = tiny || ((unsigned)x * 2u - 2u < 2u * 0x0D800000u - 2u) || ((unsigned)(x >> 32) * 2u - 2u < 2u * 0x0D800000u - 2u);
    }
    const u64 bound = f2_sub(f2_mul(k.ten, C, k.nz), f2_mul(k.nine, UU, k.nz));
    float b0, b1, Cm0, Cm1, Dm0, Dm1;
    f2_unpack(bound, b0, b1);
    f2_unpack(C, Cm0, Cm1);
    f2_unpack(D, Dm0, Dm1);
    const float lim0 = cd_limit_rising(phi30, Cm0, Dm0, b0);
    const float lim1 = cd_limit_rising(phi31, Cm1, Dm1, b1);
    const u64 cen = f2_mul(k.half, f2_add(C, D), k.nz);
    float cen0, cen1;
    f2_unpack(cen, cen0, cen1);
    const u64 phi = f2_mul(sg, f2_pack(cd_bitsel(have0, lim0, cen0), cd_bitsel(have1, lim1, cen1)), k.nz);
    const u64 F = f2_sub(f2_mul(U, phi, k.nz), f2_mul(k.nu, f2_sub(p0, m1), k.nz));
    float F0, F1;
    f2_unpack(F, F0, F1);
    f0 = cd_bitsel(wall, 0.0f, F0);
    f1 = cd_bitsel(wall, 0.0f, F1);
}

// ---- any shape ------------------------------------------------------------------------------------------------------------
// value of component c at K (K_c = N_c: the unstored upper wall, 0); caller guarantees 0 <= K_a <= N_a - 1 (a != c), 0 <= K_c <= N_c
template <typename T, int ND>
__device__ __forceinline__ T cd_at(const Grid& g, const T* __restrict__ u, int c, const int* K) {
    const int N[3] = {g.N0, g.N1, g.N2};
    if (K[c] == N[c]) return T(0);
    return u[(long long)c * g.M + cell_index(g, K[0], K[1], ND == 3 ? K[2] : 0)];
}

// F_ij at I, straight from global memory.
template <typename T, int ND>
__device__ __forceinline__ T cd_flux_at(const Grid& g, const T* __restrict__ u, T nu, int i, int j, const int* I) {
    const int N[3] = {g.N0, g.N1, g.N2};
    if (j != i && (I[j] == 0 || I[j] == N[j])) return T(0);
    int K[3] = {I[0], I[1], I[2]};
    const T a = cd_at<T, ND>(g, u, j, K);
    K[i] -= 1;
    const T b = cd_at<T, ND>(g, u, j, K);
    K[i] += 1;
    const T p0 = cd_at<T, ND>(g, u, i, K);
    K[j] -= 1;
    const T m1 = cd_at<T, ND>(g, u, i, K);
    const int top = (j == i) ? N[j] : N[j] - 1;   // last index of component i along j that holds a value
    const bool hm2 = I[j] - 2 >= 0;
    const bool hp1 = I[j] + 1 <= top;
    T m2 = T(0), p1 = T(0);
    if (hm2) { K[j] = I[j] - 2; m2 = cd_at<T, ND>(g, u, i, K); }
    if (hp1) { K[j] = I[j] + 1; p1 = cd_at<T, ND>(g, u, i, K); }
    bool tiny = false;
    typedef typename CdMask<T>::type Mk;
    return cd_flux<T, true>(a, b, m2, m1, p0, p1, hm2 ? ~Mk(0) : Mk(0), hp1 ? ~Mk(0) : Mk(0), Mk(0), nu, tiny);
}

template <typename T, int ND>
__global__ void k_convdiff(Grid g, const T* __restrict__ u, T nu, T* __restrict__ r) {
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < g.M; e += (long long)gridDim.x * blockDim.x) {
        int I[3];
        decompose<T, ND>(g, e, I[0], I[1], I[2]);
#pragma unroll
        for (int i = 0; i < ND; ++i) {
            T s = T(0);
            if (I[i] > 0) {
#pragma unroll
                for (int j = 0; j < ND; ++j) {
                    int Iu[3] = {I[0], I[1], I[2]};
                    Iu[j] += 1;
                    const T Fl = cd_flux_at<T, ND>(g, u, nu, i, j, I);
                    const T Fu = cd_flux_at<T, ND>(g, u, nu, i, j, Iu);
                    s = s + (Fl - Fu);
                }
            }
            r[(long long)i * g.M + e] = s;
        }
    }
}

// ---- 3-D, tiled ------------------------------------------------------------------------------------------------------------
template <typename T, int TY_>
struct CD3 {
    static constexpr int VEC = 16 / (int)sizeof(T);
    static constexpr int TX = 32 * VEC;          // one warp = one row of the tile
    static constexpr int TY = TY_;
    static constexpr int WX = TX + 2 * VEC;      // box: VEC cells of halo on either side (the box starts on a 16-byte boundary)
    static constexpr int WY = TY + 4;            // rows Y0-2 .. Y0+TY+1 (row Y0+TY is the flux-only row)
    static constexpr int NW = TY + 1;            // warps: TY rows that own cells + one that only evaluates the y-fluxes of row TY
    static constexpr int NT = 32 * NW;
    static constexpr int NSLOT = 6;              // ring of planes: k-2 .. k+1 (the z-window is read from here), two in flight
    static constexpr int PLANE = (WX * WY + 31) / 32 * 32;   // elements of one component in a slot (TMA destinations: 128-byte aligned)
    static constexpr int SLOT = 3 * PLANE;
    static constexpr int FROW = TX;              // flux exchange: [2 buffers][3 components][NW rows][TX]
    static constexpr int FBUF = 3 * NW * FROW;
    static constexpr int PARK = 3 * VEC * NT;    // per-thread parking of the carried z-fluxes
    static constexpr size_t smem_bytes() { return (size_t)(NSLOT * SLOT + 2 * FBUF + PARK) * sizeof(T) + 128 + (NSLOT + 1) * 8; }
};

template <typename T>
struct CdParams {
    int N0, N1, N2;
    int ntx, nty;      // tiles in x and y
    int nz;            // planes per z-chunk
    T nu;
    T* r;
    long long M;
    unsigned long long negzero2;   // two -0.0f: the addend that turns fma.rn.f32x2 into a product (wl_fused3d.cuh)
};

template <typename T, int V> struct CdVec;
template <> struct CdVec<float, 4> { typedef float4 type; };
template <> struct CdVec<double, 2> { typedef double2 type; };

template <typename T, int TY>
__global__ void __launch_bounds__(CD3<T, TY>::NT, 1)
k_convdiff3d(const __grid_constant__ CUtensorMap m0, const __grid_constant__ CUtensorMap m1, const __grid_constant__ CUtensorMap m2,
             const CdParams<T> prm) {
    using G = CD3<T, TY>;
    constexpr int VEC = G::VEC;
    typedef typename CdVec<T, VEC>::type V;

    extern __shared__ __align__(1024) unsigned char smem_raw[];
    T* ring = reinterpret_cast<T*>(smem_raw);
    T* fbuf = ring + G::NSLOT * G::SLOT;
    const int t_park_off = (int)threadIdx.x * VEC;   // [3][NT][VEC]: conflict-free 16-byte accesses
    T* park = fbuf + 2 * G::FBUF + t_park_off;
    uint64_t* full = reinterpret_cast<uint64_t*>(fbuf + 2 * G::FBUF + G::PARK);
    uint64_t* stepbar = full + G::NSLOT;

    const int t = threadIdx.x, lane = t & 31, w = t >> 5;
    // item: chunk-major, so that CTAs resident together sweep neighbouring tiles of one z-range (halo reuse in L2)
    const int tiles = prm.ntx * prm.nty;
    const int chunk = blockIdx.x / tiles;
    const int tile = blockIdx.x - chunk * tiles;
    const int ty = tile / prm.ntx, tx = tile - ty * prm.ntx;
    const int X0 = tx * G::TX, Y0 = ty * G::TY;
    const int z0 = chunk * prm.nz;
    const int z1 = min(z0 + prm.nz, prm.N2);     // planes [z0, z1) are this item's
    const int N0 = prm.N0, N1 = prm.N1, N2 = prm.N2;
    const T nu = prm.nu;

    if (t == 0) {
#pragma unroll
        for (int s = 0; s < G::NSLOT; ++s) mbar_init(&full[s], 1);
        mbar_init(stepbar, G::NW);
        fence_mbar_init();
    }
    __syncthreads();

    // plane q (z0-2 <= q <= z1+1) lives in slot (q - (z0-2)) mod NSLOT
    const int qlast = z1 + 1;
    auto issue = [&](int q) {
        const int s = (q - (z0 - 2)) % G::NSLOT;
        T* dst = ring + s * G::SLOT;
        mbar_expect_tx(&full[s], (uint32_t)(3 * G::WX * G::WY * sizeof(T)));
        tma_load_3d(dst, &m0, X0 - VEC, Y0 - 2, q, &full[s]);
        tma_load_3d(dst + G::PLANE, &m1, X0 - VEC, Y0 - 2, q, &full[s]);
        tma_load_3d(dst + 2 * G::PLANE, &m2, X0 - VEC, Y0 - 2, q, &full[s]);
    };
    if (t == 0) {
#pragma unroll
        for (int d = 0; d < G::NSLOT; ++d)
            if (z0 - 2 + d <= qlast) issue(z0 - 2 + d);
    }

    const int yy = w + 2;                 // row of the box this thread's vector sits in
    const int xx = VEC + lane * VEC;      // column
    const int gx = X0 + lane * VEC, gy = Y0 + w;
    const int own = yy * G::WX + xx;
    const bool full_row = w < TY;         // owns cells (the last warp only evaluates y-fluxes)
    const bool stores = full_row && gx < N0 && gy < N1;
    const bool live_y = gx < N0 && gy <= N1;          // this thread's y-fluxes are used by somebody

    // per-thread boundary masks.  x: only the first two and the last two flux positions of a row can lie at a wall, so the
    // masks of the other positions are compile-time constants.  y: one set per row.
    typedef typename CdMask<T>::type Mk;
    constexpr Mk kAll = ~Mk(0), kNone = Mk(0);
    const Mk xl_in = (gx == 0) ? kNone : kAll;            // false where this vector starts at the lower x-wall
    const Mk xr_in = (gx + VEC == N0) ? kNone : kAll;     // false where it ends at the upper x-wall
    const Mk wally = (gy == 0 || gy == N1) ? kAll : kNone;
    const Mk hm2y = (gy - 2 >= 0) ? kAll : kNone;
    const Mk hp1y1 = (gy + 1 <= N1) ? kAll : kNone, hp1y = (gy + 1 <= N1 - 1) ? kAll : kNone;
    const bool y_interior = gy >= 2 && gy + 1 <= N1 - 1;   // warp-uniform: no wall within reach of this row's y-fluxes
    CdConst2 k2;
    if constexpr (VEC == 4) {
        k2.half = f2_pack(0.5f, 0.5f); k2.two = f2_pack(2.0f, 2.0f); k2.five = f2_pack(5.0f, 5.0f); k2.six_neg = f2_pack(-6.0f, -6.0f);
        k2.nine = f2_pack(9.0f, 9.0f); k2.ten = f2_pack(10.0f, 10.0f);
        k2.y = f2_pack(0.16666667163372039794921875f, 0.16666667163372039794921875f);
        k2.nu = f2_pack((float)prm.nu, (float)prm.nu); k2.nz = prm.negzero2;
    }

    T acc[3][VEC];        // plane k-1: 0 + (x-flux difference) + (y-flux difference), in that order
    auto ldv = [&](const T* p, T* out) {
        const V v = *reinterpret_cast<const V*>(p);
        if constexpr (VEC == 4) { out[0] = v.x; out[1] = v.y; out[2] = v.z; out[3] = v.w; }
        else { out[0] = v.x; out[1] = v.y; }
    };
    auto ld2 = [&](const T* p, T* out) {   // two consecutive elements, 2·sizeof(T)-aligned
        if constexpr (VEC == 4) { const float2 v = *reinterpret_cast<const float2*>(p); out[0] = v.x; out[1] = v.y; }
        else { const double2 v = *reinterpret_cast<const double2*>(p); out[0] = v.x; out[1] = v.y; }
    };
    auto stv = [&](T* p, const T* in) {
        V v;
        if constexpr (VEC == 4) { v.x = in[0]; v.y = in[1]; v.z = in[2]; v.w = in[3]; }
        else { v.x = in[0]; v.y = in[1]; }
        *reinterpret_cast<V*>(p) = v;
    };

    // prologue: planes z0-2, z0-1, z0 have landed
#pragma unroll
    for (int d = 0; d < 3; ++d) mbar_wait(&full[d], 0);
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int e = 0; e < VEC; ++e) acc[c][e] = T(0);

    // One plane step per iteration.  The thread's z-window (its own vector on planes k-2 .. k+1) is read from the ring where it
    // is needed instead of being carried in registers (36 registers and as many moves per step less; carrying it was measured:
    // spills under the 168-register cap of 12 warps).
    constexpr int Wm2 = 0, Wm1 = 1, W0 = 2, Wp1 = 3;
    int s0 = 2, sp1 = 3;            // slots of planes k and k+1
    uint32_t php1 = 0;              // phase of plane k+1's slot
#pragma unroll 1
    for (int k = z0; k <= z1; ++k) {
        mbar_wait(&full[sp1], php1);
        const int sm1 = (s0 == 0) ? G::NSLOT - 1 : s0 - 1;
        const int sm2 = (sm1 == 0) ? G::NSLOT - 1 : sm1 - 1;
        const T* pk = ring + s0 * G::SLOT;              // plane k: own values and in-plane neighbours
        const T* pkm1 = ring + sm1 * G::SLOT;
        const T* pkm2 = ring + sm2 * G::SLOT;
        const T* pkp1 = ring + sp1 * G::SLOT;
        T win[3][4][VEC];
#pragma unroll
        for (int c = 0; c < 3; ++c) ldv(pk + c * G::PLANE + own, win[c][W0]);
        T* fb = fbuf + (k & 1) * G::FBUF;

        const bool inplane = k < z1;                    // the step past the chunk only needs the z-fluxes
        const Mk wallz = (k == 0 || k == N2) ? kAll : kNone;
        const Mk hm2z = (k - 2 >= 0) ? kAll : kNone;
        const Mk hp1z2 = (k + 1 <= N2) ? kAll : kNone, hp1z = (k + 1 <= N2 - 1) ? kAll : kNone;
        const bool z_interior = k >= 2 && k + 1 <= N2 - 1;

        if (inplane) {
            // y-fluxes: advecting velocity u1 at I and at I - d_i
            T fy[3][VEC];       // lower y-fluxes: parked in the exchange buffer, read back when the step's sums are formed
            T ym2[3][VEC], ym1[3][VEC], yp1[3][VEC];    // rows gy-2, gy-1, gy+1
            T u1l[2];                                   // u1 at gx-2, gx-1
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                ldv(pk + c * G::PLANE + own - 2 * G::WX, ym2[c]);
                ldv(pk + c * G::PLANE + own - G::WX, ym1[c]);
                ldv(pk + c * G::PLANE + own + G::WX, yp1[c]);
            }
            ld2(pk + G::PLANE + own - 2, u1l);
            ldv(pkm1 + G::PLANE + own, win[1][Wm1]);
            auto yflux = [&](auto EX_, auto IN_) {
                constexpr bool EX = decltype(EX_)::value;
                constexpr bool IN = decltype(IN_)::value;   // interior row: every flag is a compile-time constant
                const Mk hm2y_ = IN ? kAll : hm2y, hp1y_ = IN ? kAll : hp1y, hp1y1_ = IN ? kAll : hp1y1, wally_ = IN ? kNone : wally;
                bool tiny = false;
                if constexpr (VEC == 4) {
#pragma unroll
                    for (int e = 0; e < VEC; e += 2) {
                        const u64 a = f2_pack(win[1][W0][e], win[1][W0][e + 1]);
                        const u64 bl = f2_pack((e == 0) ? u1l[1] : win[1][W0][e > 0 ? e - 1 : 0], win[1][W0][e]);
                        cd_flux2<EX>(a, bl, f2_pack(ym2[0][e], ym2[0][e + 1]), f2_pack(ym1[0][e], ym1[0][e + 1]),
                                     f2_pack(win[0][W0][e], win[0][W0][e + 1]), f2_pack(yp1[0][e], yp1[0][e + 1]), hm2y_, hp1y_, wally_, k2, tiny,
                                     fy[0][e], fy[0][e + 1]);
                        cd_flux2<EX>(a, f2_pack(ym1[1][e], ym1[1][e + 1]), f2_pack(ym2[1][e], ym2[1][e + 1]), f2_pack(ym1[1][e], ym1[1][e + 1]),
                                     f2_pack(win[1][W0][e], win[1][W0][e + 1]), f2_pack(yp1[1][e], yp1[1][e + 1]), hm2y_, hp1y1_, kNone, k2, tiny,
                                     fy[1][e], fy[1][e + 1]);
                        cd_flux2<EX>(a, f2_pack(win[1][Wm1][e], win[1][Wm1][e + 1]), f2_pack(ym2[2][e], ym2[2][e + 1]), f2_pack(ym1[2][e], ym1[2][e + 1]),
                                     f2_pack(win[2][W0][e], win[2][W0][e + 1]), f2_pack(yp1[2][e], yp1[2][e + 1]), hm2y_, hp1y_, wally_, k2, tiny,
                                     fy[2][e], fy[2][e + 1]);
                    }
                } else {
#pragma unroll
                    for (int e = 0; e < VEC; ++e) {
                        const T a = win[1][W0][e];
                        const T bl = (e == 0) ? u1l[1] : win[1][W0][e > 0 ? e - 1 : 0];
                        fy[0][e] = cd_flux<T, EX>(a, bl, ym2[0][e], ym1[0][e], win[0][W0][e], yp1[0][e], hm2y_, hp1y_, wally_, nu, tiny);
                        fy[1][e] = cd_flux<T, EX>(a, ym1[1][e], ym2[1][e], ym1[1][e], win[1][W0][e], yp1[1][e], hm2y_, hp1y1_, kNone, nu, tiny);
                        fy[2][e] = cd_flux<T, EX>(a, win[1][Wm1][e], ym2[2][e], ym1[2][e], win[2][W0][e], yp1[2][e], hm2y_, hp1y_, wally_, nu, tiny);
                    }
                }
                return tiny;
            };
            if (y_interior) { if (yflux(std::false_type{}, std::true_type{}) && live_y) yflux(std::true_type{}, std::true_type{}); }
            else if (yflux(std::false_type{}, std::false_type{}) && live_y) yflux(std::true_type{}, std::false_type{});
            // hand the lower y-fluxes to the row below
#pragma unroll
            for (int c = 0; c < 3; ++c) stv(fb + (c * G::NW + w) * G::FROW + lane * VEC, fy[c]);
        }
        if (full_row) {
            {
                // z-fluxes: advecting velocity u2 at I and at I - d_i; then plane k-1 is complete: r = acc + (Fz(k-1) - Fz(k))
                T fz[3][VEC];
                T u2l[2], u2d[VEC];                     // u2 at gx-2, gx-1; u2 on row gy-1
                ld2(pk + 2 * G::PLANE + own - 2, u2l);
                ldv(pk + 2 * G::PLANE + own - G::WX, u2d);
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    ldv(pkm2 + c * G::PLANE + own, win[c][Wm2]);
                    ldv(pkm1 + c * G::PLANE + own, win[c][Wm1]);
                    ldv(pkp1 + c * G::PLANE + own, win[c][Wp1]);
                }
                auto zflux = [&](auto EX_, auto IN_) {
                    constexpr bool EX = decltype(EX_)::value;
                    constexpr bool IN = decltype(IN_)::value;   // interior plane
                    const Mk hm2z_ = IN ? kAll : hm2z, hp1z_ = IN ? kAll : hp1z, hp1z2_ = IN ? kAll : hp1z2, wallz_ = IN ? kNone : wallz;
                    bool tiny = false;
                    if constexpr (VEC == 4) {
#pragma unroll
                        for (int e = 0; e < VEC; e += 2) {
                            const u64 a = f2_pack(win[2][W0][e], win[2][W0][e + 1]);
                            const u64 bl = f2_pack((e == 0) ? u2l[1] : win[2][W0][e > 0 ? e - 1 : 0], win[2][W0][e]);
                            cd_flux2<EX>(a, bl, f2_pack(win[0][Wm2][e], win[0][Wm2][e + 1]), f2_pack(win[0][Wm1][e], win[0][Wm1][e + 1]),
                                         f2_pack(win[0][W0][e], win[0][W0][e + 1]), f2_pack(win[0][Wp1][e], win[0][Wp1][e + 1]), hm2z_, hp1z_, wallz_, k2, tiny,
                                         fz[0][e], fz[0][e + 1]);
                            cd_flux2<EX>(a, f2_pack(u2d[e], u2d[e + 1]), f2_pack(win[1][Wm2][e], win[1][Wm2][e + 1]), f2_pack(win[1][Wm1][e], win[1][Wm1][e + 1]),
                                         f2_pack(win[1][W0][e], win[1][W0][e + 1]), f2_pack(win[1][Wp1][e], win[1][Wp1][e + 1]), hm2z_, hp1z_, wallz_, k2, tiny,
                                         fz[1][e], fz[1][e + 1]);
                            cd_flux2<EX>(a, f2_pack(win[2][Wm1][e], win[2][Wm1][e + 1]), f2_pack(win[2][Wm2][e], win[2][Wm2][e + 1]), f2_pack(win[2][Wm1][e], win[2][Wm1][e + 1]),
                                         f2_pack(win[2][W0][e], win[2][W0][e + 1]), f2_pack(win[2][Wp1][e], win[2][Wp1][e + 1]), hm2z_, hp1z2_, kNone, k2, tiny,
                                         fz[2][e], fz[2][e + 1]);
                        }
                    } else {
#pragma unroll
                        for (int e = 0; e < VEC; ++e) {
                            const T a = win[2][W0][e];
                            const T bl = (e == 0) ? u2l[1] : win[2][W0][e > 0 ? e - 1 : 0];
                            fz[0][e] = cd_flux<T, EX>(a, bl, win[0][Wm2][e], win[0][Wm1][e], win[0][W0][e], win[0][Wp1][e], hm2z_, hp1z_, wallz_, nu, tiny);
                            fz[1][e] = cd_flux<T, EX>(a, u2d[e], win[1][Wm2][e], win[1][Wm1][e], win[1][W0][e], win[1][Wp1][e], hm2z_, hp1z_, wallz_, nu, tiny);
                            fz[2][e] = cd_flux<T, EX>(a, win[2][Wm1][e], win[2][Wm2][e], win[2][Wm1][e], win[2][W0][e], win[2][Wp1][e], hm2z_, hp1z2_, kNone, nu, tiny);
                        }
                    }
                    return tiny;
                };
                if (z_interior) { if (zflux(std::false_type{}, std::true_type{}) && stores) zflux(std::true_type{}, std::true_type{}); }
                else if (zflux(std::false_type{}, std::false_type{}) && stores) zflux(std::true_type{}, std::false_type{});
                if (k > z0 && stores) {
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        T o[VEC], fzp[VEC];               // lower z-flux of plane k-1, parked by the previous step
                        ldv(park + c * G::NT * VEC, fzp);
#pragma unroll
                        for (int e = 0; e < VEC; ++e) {
                            o[e] = acc[c][e] + (fzp[e] - fz[c][e]);
                            const bool wallface = (c == 0) ? (gx + e == 0) : (c == 1) ? (gy == 0) : (k - 1 == 0);
                            if (wallface) o[e] = T(0);
                        }
                        stv(prm.r + (long long)c * prm.M + ((long long)gx + (long long)N0 * ((long long)gy + (long long)N1 * (k - 1))), o);
                    }
                }
#pragma unroll
                for (int c = 0; c < 3; ++c) stv(park + c * G::NT * VEC, fz[c]);
            }
            if (inplane) {
                // x-fluxes at gx .. gx+VEC: advecting velocity u0 at I and at I - d_i.  These are the last reads of plane k.
                T ext[3][VEC + 4];                      // x-extended rows: ext[c][0..VEC+3] = cells gx-2 .. gx+VEC+1
                T u0d[VEC];                             // u0 on row gy-1
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    ld2(pk + c * G::PLANE + own - 2, &ext[c][0]);
#pragma unroll
                    for (int e = 0; e < VEC; ++e) ext[c][2 + e] = win[c][W0][e];
                    ld2(pk + c * G::PLANE + own + VEC, &ext[c][VEC + 2]);
                }
                ldv(pk + own - G::WX, u0d);
                const T u0ym1_r = pk[own - G::WX + VEC];    // u0 at (gx+VEC, gy-1)
                ldv(pkm1 + own, win[0][Wm1]);
                const T u0r_prev = pkm1[own + VEC];        // u0 at (gx+VEC, gy) on plane k-1
                __syncwarp();
                if (lane == 0) mbar_arrive(stepbar);
                auto xflux = [&](auto EX_) {
                    constexpr bool EX = decltype(EX_)::value;
                    bool tiny = false;
                    T fx[3][VEC + 1];
#pragma unroll
                    for (int e = 0; e <= VEC; ++e) {
                        const Mk h2 = (e < 2) ? xl_in : kAll;                         // gx+e-2 >= 0
                        const Mk h10 = (e == VEC) ? xr_in : kAll;                     // gx+e+1 <= N0     (component 0 holds the wall value at N0)
                        const Mk h1 = (e >= VEC - 1) ? xr_in : kAll;                  // gx+e+1 <= N0 - 1
                        const Mk wl_ = (e == 0) ? ~xl_in : (e == VEC) ? ~xr_in : kNone;   // gx+e == 0 or N0
                        const T a = ext[0][2 + e];
                        const T b1 = (e < VEC) ? u0d[e < VEC ? e : 0] : u0ym1_r;
                        const T b2 = (e < VEC) ? win[0][Wm1][e < VEC ? e : 0] : u0r_prev;
                        fx[0][e] = cd_flux<T, EX>(a, ext[0][1 + e], ext[0][e], ext[0][1 + e], ext[0][2 + e], ext[0][3 + e], h2, h10, kNone, nu, tiny);
                        fx[1][e] = cd_flux<T, EX>(a, b1, ext[1][e], ext[1][1 + e], ext[1][2 + e], ext[1][3 + e], h2, h1, wl_, nu, tiny);
                        fx[2][e] = cd_flux<T, EX>(a, b2, ext[2][e], ext[2][1 + e], ext[2][2 + e], ext[2][3 + e], h2, h1, wl_, nu, tiny);
                    }
#pragma unroll
                    for (int c = 0; c < 3; ++c)
#pragma unroll
                        for (int e = 0; e < VEC; ++e) acc[c][e] = T(0) + (fx[c][e] - fx[c][e + 1]);
                    return tiny;
                };
                if (xflux(std::false_type{}) && stores) xflux(std::true_type{});
            }
        } else if (inplane) {
            __syncwarp();
            if (lane == 0) mbar_arrive(stepbar);
        }
        if (inplane) {
            // everybody's y-fluxes of this plane are in fb, and nobody reads plane k-2 any more
            mbar_wait(stepbar, (uint32_t)((k - z0) & 1));
            if (t == 0 && k + 4 <= qlast) issue(k + 4);
            if (full_row) {
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    T fl[VEC], fu[VEC];
                    ldv(fb + (c * G::NW + w) * G::FROW + lane * VEC, fl);
                    ldv(fb + (c * G::NW + w + 1) * G::FROW + lane * VEC, fu);
#pragma unroll
                    for (int e = 0; e < VEC; ++e) acc[c][e] = acc[c][e] + (fl[e] - fu[e]);
                }
            }
        }
        s0 = sp1;
        sp1 = (sp1 + 1 == G::NSLOT) ? 0 : sp1 + 1;
        if (sp1 == 0) php1 ^= 1u;
    }
}

}  // namespace wl
