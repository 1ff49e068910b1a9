// wl_rates.cuh — device self-measurement of the fp32 arithmetic rate of one SM: scalar against packed (f32x2) add and fma.
//
// The fused kernels and wl_convdiff use add/sub/mul.rn.f32x2 (FADD2 / FFMA2).  Whether a packed instruction doubles the
// arithmetic per clock or only halves the issue slots decides the ALU ceiling bench.py divides wl_convdiff by
// (DESIGN.md §6.6).  Measured here with clock64 around a long unrolled loop of independent chains, 16 warps per SM, one CTA
// per SM.  Result on B200 (profiles/r3_packed_rate.md): 3.95 scalar and 2.00 packed warp-instructions per clock and SM, i.e.
// 128 lane-operations per clock and SM either way — a packed instruction holds the FMA pipe twice as long.
#pragma once
#include "wl_common.cuh"

namespace wl {

// MODE 0: add.rn.f32, 1: add.rn.f32x2, 2: fma.rn.f32, 3: fma.rn.f32x2.  cyc[blockIdx.x] = clocks of the timed loop.
template <int MODE>
__global__ void __launch_bounds__(512) k_fp32_rate(float* sink, long long* cyc, int iters, float seed) {
    float a[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) a[i] = seed * (float)(i + 1) + (float)threadIdx.x;
    const float inc = seed * 0.5f;
    unsigned long long inc2;
    asm("mov.b64 %0, {%1, %1};" : "=l"(inc2) : "f"(inc));
    __syncthreads();
    const long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
        if (MODE == 0 || MODE == 2) {
#pragma unroll
            for (int i = 0; i < 16; ++i) {
                if (MODE == 0) asm volatile("add.rn.f32 %0, %0, %1;" : "+f"(a[i]) : "f"(inc));
                else asm volatile("fma.rn.f32 %0, %0, %1, %1;" : "+f"(a[i]) : "f"(inc));
            }
        } else {
#pragma unroll
            for (int i = 0; i < 16; i += 2) {
                unsigned long long v;
                asm("mov.b64 %0, {%1, %2};" : "=l"(v) : "f"(a[i]), "f"(a[i + 1]));
                if (MODE == 1) asm volatile("add.rn.f32x2 %0, %0, %1;" : "+l"(v) : "l"(inc2));
                else asm volatile("fma.rn.f32x2 %0, %0, %1, %1;" : "+l"(v) : "l"(inc2));
                asm("mov.b64 {%0, %1}, %2;" : "=f"(a[i]), "=f"(a[i + 1]) : "l"(v));
            }
        }
    }
    const long long t1 = clock64();
    float s = 0;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += a[i];
    if (s == 123.456f) sink[0] = s;   // keeps the chains alive; practically never taken
    if (threadIdx.x == 0) cyc[blockIdx.x] = t1 - t0;
}

}  // namespace wl
