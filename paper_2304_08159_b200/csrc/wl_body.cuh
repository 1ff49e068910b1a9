// wl_body.cuh — BDIM face coefficients from analytic bodies, on the device (the `BDIM!` row of the
// paper's Table 2; "the immersed geometry from a user-defined signed-distance function").
//
//   L[i][I] = mu0(d),  d = min over bodies of the signed distance (in cells, positive in the fluid) at the CENTRE of face
//   (I,i): coordinate I_i along i, I_j + 1/2 along every other axis;
//   mu0(d) = 0 for d <= -1, 1 for d >= 1, else 0.5 (1 + d + sin(pi d)/pi), evaluated in fp64, clamped to [0,1], THEN cast
//   to T (c-8: BJ "BDIM face coefficient");  the stored wall plane I_i = 0 is 0 (BJ "zero on domain-boundary faces").
//
// One launch writes the context's level-0 coefficient array; the coarsening chain of wl_set_coeff follows.  A moving body
// costs this kernel per step instead of an upload of n·M coefficients.  Row-wise, 16-byte stores; a body whose bounding
// tube (radius + 2 cells) misses the row is rejected once per row.
#pragma once
#include "wl_common.cuh"
#include "wl_fused3d.cuh"   // st_vec
#include "wl_rows.cuh"      // kRowsX, kRowsY

namespace wl {

constexpr int kBodyDoubles = 8;    // per body: kind, c0, c1, c2, R, r, 0, 0
constexpr int kMaxBodies = 256;

__device__ __forceinline__ double mu0_device(double d) {
    if (d <= -1.0) return 0.0;
    if (d >= 1.0) return 1.0;
    const double kPi = 3.14159265358979323846;
    double v = 0.5 * (1.0 + d + sin(kPi * d) / kPi);
    v = fmin(fmax(v, 0.0), 1.0);
    return v;
}

template <typename T, int ND>
__global__ void __launch_bounds__(kRowsX* kRowsY) k_body_coeff_rows(Grid g, const double* __restrict__ bodies, int nbodies,
                                                                   T* __restrict__ Lout) {
    constexpr int VEC = 16 / (int)sizeof(T);
    __shared__ double sb[kMaxBodies * kBodyDoubles];
    for (int i = threadIdx.y * kRowsX + threadIdx.x; i < nbodies * kBodyDoubles; i += kRowsX * kRowsY) sb[i] = bodies[i];
    __syncthreads();
    const int nvx = g.N0 / VEC;
    const long long rows_per_comp = (long long)g.N1 * g.N2;
    const long long nrows = rows_per_comp * ND;
    for (long long r = (long long)blockIdx.x * kRowsY + threadIdx.y; r < nrows; r += (long long)gridDim.x * kRowsY) {
        const int comp = (int)(r / rows_per_comp);
        const long long rc = r - (long long)comp * rows_per_comp;
        const int z = (int)(rc / g.N1), y = (int)(rc - (long long)z * g.N1);
        const bool wall_row = (comp == 1 && y == 0) || (comp == 2 && z == 0);
        const double fy = (double)y + (comp == 1 ? 0.0 : 0.5);
        const double fz = (ND == 3) ? (double)z + (comp == 2 ? 0.0 : 0.5) : 0.0;
        T* dst = Lout + r * g.N0;
        for (int vx = threadIdx.x; vx < nvx; vx += kRowsX) {
            double dmin[VEC];
#pragma unroll
            for (int k = 0; k < VEC; ++k) dmin[k] = 1.0e300;
            if (!wall_row) {
                for (int bi = 0; bi < nbodies; ++bi) {
                    const double* B = sb + bi * kBodyDoubles;
                    const int kind = (int)B[0];
                    const double dy = fy - B[2], dz = (ND == 3) ? fz - B[3] : 0.0;
                    const double R = B[4], rr = B[5];
                    if (kind == 0) {            // sphere (circle in 2-D): d = |x - c| - R
                        const double reach = R + 2.0;
                        if (dy * dy + dz * dz >= reach * reach) continue;
#pragma unroll
                        for (int k = 0; k < VEC; ++k) {
                            const double dx = ((double)(vx * VEC + k) + (comp == 0 ? 0.0 : 0.5)) - B[1];
                            double r2 = dx * dx + dy * dy;
                            if (ND == 3) r2 = r2 + dz * dz;
                            dmin[k] = fmin(dmin[k], sqrt(r2) - R);
                        }
                    } else {                    // torus about axis 0: d = sqrt((sqrt(y^2 + z^2) - R)^2 + x^2) - r
                        const double rho = sqrt(dy * dy + dz * dz) - R;
                        if (fabs(rho) >= rr + 2.0) continue;
#pragma unroll
                        for (int k = 0; k < VEC; ++k) {
                            const double dx = ((double)(vx * VEC + k) + (comp == 0 ? 0.0 : 0.5)) - B[1];
                            dmin[k] = fmin(dmin[k], sqrt(rho * rho + dx * dx) - rr);
                        }
                    }
                }
            }
            T v[VEC];
#pragma unroll
            for (int k = 0; k < VEC; ++k) v[k] = wall_row ? (T)0 : (T)mu0_device(dmin[k]);
            if (comp == 0 && vx == 0) v[0] = (T)0;
            st_vec<T, VEC>(dst + vx * VEC, v);
        }
    }
}

// Any-shape version (rows that are not whole 16-byte vectors): one thread per face.
template <typename T, int ND>
__global__ void k_body_coeff(Grid g, const double* __restrict__ bodies, int nbodies, T* __restrict__ Lout) {
    const long long total = g.M * ND;
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (long long)gridDim.x * blockDim.x) {
        const int comp = (int)(e / g.M);
        const long long I = e - (long long)comp * g.M;
        int i0, i1, i2;
        decompose<T, ND>(g, I, i0, i1, i2);
        const int Ii[3] = {i0, i1, i2};
        if (Ii[comp] == 0) { Lout[e] = (T)0; continue; }
        const double fx = (double)i0 + (comp == 0 ? 0.0 : 0.5), fy = (double)i1 + (comp == 1 ? 0.0 : 0.5);
        const double fz = (ND == 3) ? (double)i2 + (comp == 2 ? 0.0 : 0.5) : 0.0;
        double dmin = 1.0e300;
        for (int bi = 0; bi < nbodies; ++bi) {
            const double* B = bodies + bi * kBodyDoubles;
            const double dx = fx - B[1], dy = fy - B[2], dz = (ND == 3) ? fz - B[3] : 0.0;
            if ((int)B[0] == 0) {
                double r2 = dx * dx + dy * dy;
                if (ND == 3) r2 = r2 + dz * dz;
                dmin = fmin(dmin, sqrt(r2) - B[4]);
            } else {
                const double rho = sqrt(dy * dy + dz * dz) - B[4];
                dmin = fmin(dmin, sqrt(rho * rho + dx * dx) - B[5]);
            }
        }
        Lout[e] = (T)mu0_device(dmin);
    }
}

}  // namespace wl
