// wl_static.cu — wl_residual_norm_static: the residual check of include/wl.h for callers that cannot allocate device memory.
//
// Who that is.  A flow solver that sized its velocity, pressure and coefficient arrays to fill the GPU when it started has
// nothing left for cudaMalloc to hand out in the middle of a run; a host framework that took all of device memory into its
// own pool gives a plug-in no raw allocator at all; and a time-step loop that shares the GPU with other streams cannot
// afford cudaMalloc / cudaFree there because both stall the whole device until it is idle.  Every other entry point of
// this library goes through a wl_ctx, and wl_create (and some first calls) allocate.  This one needs no context: the
// caller passes the inputs and the output, and the only extra global memory the kernel touches — one partial sum per CTA,
// the running maximum and the CTA ticket — lives in the file-scope array below, which is part of the library image.
//
// Cost and limits of that choice, for the user:
//   * every GPU that loads libwl.so holds kScratchBytes (about 128 KiB) until the process exits, used or not;
//   * one partial per 8192 cells fixes the largest grid at WL_STATIC_MAX_CELLS = 2^27 cells (512^3); larger grids are
//     refused with WL_EDIMS, nothing is launched;
//   * all calls on one device share the array.  It still holds the previous call's contents when the next one starts, so
//     each call clears the part that must start at zero (maximum, ticket) on the caller's stream before its kernel; the
//     partials need no clearing because a call reads back only the entries it wrote itself.  Two calls that are in flight
//     on the same GPU at the same time (different streams, different host threads) race on it: keep them on one stream
//     or order them with events;
//   * the device address of the array is looked up once per device, by the first call made while that device is
//     current.  That first call also makes the CUDA runtime load this module on the device, so make it during start-up,
//     before any stream capture begins.
//
// In host code the name g_static_scratch is only a handle for the symbol — it is not a device address, and a kernel handed
// `g_static_scratch` from the host side would fault or scribble over whatever host page it aliases.  The address comes
// from cudaGetSymbolAddress, with the owning device current, and that is what the kernel receives.
//
// No cudaMalloc, cudaFree, cudaMallocAsync or allocating library call anywhere in this file.
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <mutex>

#include "../../include/wl.h"
#include "wl_common.cuh"

using namespace wl;

namespace {

constexpr int kThreads = 256;
constexpr int kCellsPerThread = 32;
constexpr long long kCellsPerCta = (long long)kThreads * kCellsPerThread;                  // 8192
constexpr long long kMaxCells = WL_STATIC_MAX_CELLS;                                       // 2^27
constexpr int kMaxCtas = (int)((kMaxCells + kCellsPerCta - 1) / kCellsPerCta);             // 16384 partials
constexpr size_t kHeaderBytes = 256;                                                       // maximum + ticket, padded
constexpr size_t kScratchBytes = kHeaderBytes + sizeof(double) * (size_t)kMaxCtas;         // 131 328 bytes

struct StaticHeader {
    unsigned long long absmax_bits;   // bit pattern of max |b - A p| so far (non-negative doubles order like integers)
    unsigned int ticket;              // CTAs of the running launch that have finished
};
static_assert(sizeof(StaticHeader) <= kHeaderBytes, "header must fit its slot");

// The scratch itself.  Lives in every GPU that loads the library, from module load until the process exits.
static __device__ __align__(256) unsigned char g_static_scratch[kScratchBytes];

// ||b - A p||inf and mean(p) of one grid in ONE launch.  CTA c owns cells [c * 8192, (c+1) * 8192); the operator is the one
// of include/wl.h ("Operator"), evaluated in the term order of the library's other residual kernels, so the norm is the
// same number they produce.  The last CTA to finish (ticket) adds the per-CTA sums in a fixed order — the mean does not
// depend on scheduling — and writes both results.
template <typename T, int ND>
__global__ void __launch_bounds__(kThreads)
k_resnorm_static(Grid g, const T* __restrict__ L, const T* __restrict__ p, const T* __restrict__ b, unsigned char* scratch,
                 double* __restrict__ out) {
    __shared__ double red[32];
    __shared__ int is_last;
    StaticHeader* hdr = (StaticHeader*)scratch;
    double* partials = (double*)(scratch + kHeaderBytes);
    const int Ni[3] = {g.N0, g.N1, g.N2};
    const long long st[3] = {1, (long long)g.N0, (long long)g.N0 * g.N1};
    const long long base = (long long)blockIdx.x * kCellsPerCta;
    double m = 0.0, s = 0.0;
#pragma unroll 4
    for (int k = 0; k < kCellsPerThread; ++k) {
        const long long I = base + (long long)k * kThreads + threadIdx.x;
        if (I >= g.M) break;
        const long long q = I / g.N0;
        int Ii[3];
        Ii[0] = (int)(I - q * g.N0);
        if (ND == 3) {
            const long long q2 = q / g.N1;
            Ii[1] = (int)(q - q2 * g.N1);
            Ii[2] = (int)q2;
        } else {
            Ii[1] = (int)q;
            Ii[2] = 0;
        }
        const T pc = p[I];
        T Ax = 0;
#pragma unroll
        for (int i = 0; i < ND; ++i) {
            const T* Li = L + (long long)i * g.M;
            if (Ii[i] + 1 < Ni[i]) Ax += Li[I + st[i]] * (p[I + st[i]] - pc);   // upper face; the wall I_i = N_i is not stored
            if (Ii[i] > 0) Ax += Li[I] * (p[I - st[i]] - pc);                   // lower face; the wall plane I_i = 0 is never read
        }
        m = nanmax(m, fabs((double)(b[I] - Ax)));
        s += (double)pc;
    }
    m = block_max(m, red);
    s = block_sum(s, red);
    if (threadIdx.x == 0) {
        atomic_max_nonneg(&hdr->absmax_bits, m);
        partials[blockIdx.x] = s;
        __threadfence();                                            // partial and maximum visible before the ticket
        is_last = (atomicAdd(&hdr->ticket, 1u) == gridDim.x - 1) ? 1 : 0;
    }
    __syncthreads();
    if (is_last && threadIdx.x < 32) {
        __threadfence();
        const double total = ordered_sum(partials, (int)gridDim.x, 1);
        if (threadIdx.x == 0) {
            out[0] = __longlong_as_double((long long)*((volatile unsigned long long*)&hdr->absmax_bits));
            out[1] = total / (double)g.M;
        }
    }
}

// ---- host side ---------------------------------------------------------------------------------------------------------
constexpr int kMaxDevices = 64;
std::mutex g_mu;
unsigned char* g_scratch_addr[kMaxDevices] = {};   // device address of g_static_scratch on device d (nullptr: not looked up yet)
thread_local char g_err[256] = "";

int fail_static(int code, const char* what, cudaError_t e = cudaSuccess) {
    if (e != cudaSuccess) snprintf(g_err, sizeof(g_err), "wl_residual_norm_static: %s: %s", what, cudaGetErrorString(e));
    else snprintf(g_err, sizeof(g_err), "wl_residual_norm_static: %s", what);
    return code;
}

// Device address of the scratch array on the CURRENT device; looked up on the first call per device.
int scratch_for_current_device(unsigned char** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail_static(WL_ECUDA, "cudaGetDevice", e);
    if (dev < 0 || dev >= kMaxDevices) return fail_static(WL_ECUDA, "device ordinal beyond the table of this entry point");
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_scratch_addr[dev]) {
        unsigned char* ptr = nullptr;
        e = cudaGetSymbolAddress((void**)&ptr, g_static_scratch);   // `dev` is current here: the address belongs to it
        if (e != cudaSuccess || !ptr) return fail_static(WL_ECUDA, "cudaGetSymbolAddress(g_static_scratch)", e);
        g_scratch_addr[dev] = ptr;
    }
    *out = g_scratch_addr[dev];
    return WL_OK;
}

template <typename T>
cudaError_t launch_static(const Grid& g, const void* L, const void* p, const void* b, unsigned char* scratch, double* out,
                          cudaStream_t stream) {
    const int grid = (int)((g.M + kCellsPerCta - 1) / kCellsPerCta);
    if (g.n == 3)
        k_resnorm_static<T, 3><<<grid, kThreads, 0, stream>>>(g, (const T*)L, (const T*)p, (const T*)b, scratch, out);
    else
        k_resnorm_static<T, 2><<<grid, kThreads, 0, stream>>>(g, (const T*)L, (const T*)p, (const T*)b, scratch, out);
    return cudaGetLastError();
}

}  // namespace

extern "C" {

int wl_residual_norm_static(int ndim, const int64_t* dims, int dtype, const void* L_dev, const void* p_dev, const void* b_dev,
                            double* out_dev, void* cuda_stream) {
    g_err[0] = 0;
    if (!dims || !L_dev || !p_dev || !b_dev || !out_dev) return fail_static(WL_EINVAL, "null pointer");
    if (dtype != WL_F32 && dtype != WL_F64) return fail_static(WL_EINVAL, "dtype must be WL_F32 or WL_F64");
    if (((uintptr_t)out_dev & 7) != 0) return fail_static(WL_EINVAL, "out_dev must be 8-byte aligned");
    if (ndim != 2 && ndim != 3) return fail_static(WL_EDIMS, "ndim must be 2 or 3");
    long long M = 1;
    for (int i = 0; i < ndim; ++i) {
        if (dims[i] < 4 || dims[i] > kMaxCells) return fail_static(WL_EDIMS, "every extent must be in [4, WL_STATIC_MAX_CELLS]");
        M *= (long long)dims[i];
        if (M > kMaxCells) {
            snprintf(g_err, sizeof(g_err),
                     "wl_residual_norm_static: grid exceeds WL_STATIC_MAX_CELLS = %lld cells (the static scratch holds one partial "
                     "per %lld cells); use wl_residual_norm on a context instead", kMaxCells, kCellsPerCta);
            return WL_EDIMS;
        }
    }
    Grid g;
    g.n = ndim;
    g.N0 = (int)dims[0];
    g.N1 = (int)dims[1];
    g.N2 = ndim == 3 ? (int)dims[2] : 1;
    g.M = M;

    unsigned char* scratch = nullptr;
    int rc = scratch_for_current_device(&scratch);
    if (rc) return rc;
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    // The array still holds the last call's maximum and a full ticket: clear them, in stream order, before the kernel.
    cudaError_t e = cudaMemsetAsync(scratch, 0, kHeaderBytes, stream);
    if (e != cudaSuccess) return fail_static(WL_ECUDA, "cudaMemsetAsync(header)", e);
    e = dtype == WL_F32 ? launch_static<float>(g, L_dev, p_dev, b_dev, scratch, out_dev, stream)
                        : launch_static<double>(g, L_dev, p_dev, b_dev, scratch, out_dev, stream);
    if (e != cudaSuccess) return fail_static(WL_ECUDA, "kernel launch", e);
    return WL_OK;
}

const char* wl_static_last_error(void) { return g_err; }

}  // extern "C"
