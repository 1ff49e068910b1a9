// wl_api.cu — context, level hierarchy, launch sequencing and the C ABI of include/wl.h.
//
// Runtime structure: one context per grid; the context owns every coarse level (L, x ping-pong, b),
// a level-0 ping-pong buffer, the device scalars (norms, mean, stop flag), and the captured V-cycle graph.
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>
#include <initializer_list>
#include <math.h>
#include <new>
#include <utility>
#include <vector>

#include "../../include/wl.h"
#include "wl_common.cuh"
#include "wl_generic.cuh"
#include "wl_plan.h"
#include "wl_fused3d.cuh"
#include "wl_fused2d.cuh"
#include "wl_tail.cuh"
#include "wl_rows.cuh"
#include "wl_pcg.cuh"
#include "wl_body.cuh"
#include "wl_convdiff.cuh"
#include "wl_rates.cuh"

using namespace wl;

namespace {

// fp64 fused 3-D kernels: 1 (default) = read omega/D as a precomputed sixth plane, 0 = recompute it from the coefficients with an
// IEEE division, as the fp32 kernels do with their reciprocal.  A/B switch (build.py: WL_NVCC_EXTRA=-DWL_FP64_C_PLANE=0).  Measured
// at 256^3 on a B200 (round 3): recomputing saves 134 MB of DRAM traffic per launch but costs more than it saves — level-0 DOWN
// 0.280 ms against 0.242 ms with the plane (the division's ~20 dependent FP64 instructions, a few spilled registers), UP unchanged
// at 0.250 ms, V-cycle 0.696 against 0.643 ms — so the plane stays.
#ifndef WL_FP64_C_PLANE
#define WL_FP64_C_PLANE 1
#endif

constexpr int kMaxLevels = 32;
constexpr int kBlock = 256;
constexpr int kMaxPartials = 1 << 15;   // per-CTA sum partials (fused 2-D kernels: one per tile)
constexpr int kTailSmemBudget = 200 * 1024;

struct Level {
    Grid g;
    void* L = nullptr;      // n*M coefficients (ctx-owned copy / coarsened)
    void* C = nullptr;      // M: omega·(1/D) per cell (0 where D = 0), derived from L by wl_set_coeff; fp64 3-D contexts only
    void* x[2] = {nullptr, nullptr};  // level >= 1: iterate ping-pong; level 0: x[1] = ctx-owned scratch only
    void* b = nullptr;      // level >= 1: restricted residual
    void* tmp = nullptr;    // generic path only: second half of the Jacobi ping-pong (allocated on first use)
    int4* plan_items = nullptr;   // fused 3-D level half: per-CTA work lists (wl_plan.h), built on first use
    int* plan_start = nullptr;
    int plan_grid = 0;
};

thread_local char g_create_err[256] = "";

}  // namespace

struct wl_ctx {
    int n = 0, dtype = 0, nlev = 0;
    size_t esz = 4;
    Level lev[kMaxLevels];
    cudaStream_t stream = 0;
    Scalars* d_scal = nullptr;
    Scalars* h_scal = nullptr;   // pinned mirror
    double* d_partials = nullptr;
    double* d_hist = nullptr;
    double* h_hist = nullptr;    // pinned
    int hist_cap = 0;
    void* b0 = nullptr;          // ctx-owned right-hand side for wl_project
    double* d_bodies = nullptr;  // device copy of the body records of wl_set_bodies
    double* h_bodies = nullptr;  // pinned staging copy of the caller's records: the caller may rewrite its array as soon as the call returns
    cudaEvent_t ev_bodies = nullptr;   // the upload out of h_bodies has completed
    void* cg_v[4] = {nullptr, nullptr, nullptr, nullptr};   // r, z, p, q of the conjugate-gradient solve (allocated on first use)
    int opt_solver = 0;          // WL_OPT_SOLVER: 0 = V-cycles (BJ), 1 = V-cycle-preconditioned CG (NEXT-1)
    void* stage_u = nullptr;     // device staging for wl_project_host
    void* stage_L = nullptr;
    void* stage_p = nullptr;
    cudaStream_t copy_stream = nullptr;   // wl_project_host: copies that overlap kernels of the ctx stream
    cudaEvent_t ev_copy[3] = {nullptr, nullptr, nullptr};
    int opt_host_p_zero = 0;     // WL_OPT_HOST_P_ZERO: wl_project_host starts from p = 0 without uploading p_host
    bool have_coeff = false;
    int opt_fused = 1, opt_graph = 1, opt_coarse_cta = 1, opt_solve_kernels = 0;
    int solve_kernels_now = 0;   // WL_OPT_SOLVE_KERNELS applies to the wl_down / wl_up ENTRY POINTS only: set for the length of such a
                                 // call, so that the V-cycles of wl_vcycle / wl_solve / wl_solve_pcg never pick those instances up
    int opt_pdl = 1;             // WL_OPT_PDL: chain the cycle's kernels by programmatic dependent launch
    bool pdl_armed = false;      // the last launch enqueued by the running call was a kernel that waits before touching data
    int num_sms = 148;
    // cached CUDA graph of one V-cycle (H9), valid for one (p, b, variant, stream, options) combination
    cudaStream_t own_stream = nullptr;   // the legacy default stream cannot be captured: graphs then run here, fenced by events
    cudaEvent_t ev_in = nullptr, ev_out = nullptr;
    struct GraphEntry {          // a small LRU: a time stepper that alternates two pressure buffers, or mixes wl_vcycle with
        cudaGraphExec_t exec = nullptr;   // wl_solve, does not re-capture on every call
        void* p = nullptr;
        const void* b = nullptr;
        int variant = -1;
        int64_t nodes = 0;
        uint64_t stamp = 0;
    } cg[4];
    uint64_t cg_clock = 0;
    bool unaligned = false;      // a caller array of the running call is not 16-byte aligned: no TMA on its level
    int unaligned_level = 0;
    int tail_first = kMaxLevels; // first level of the single-CTA coarse tail (>= nlev: none fits shared memory)
    int pcg_up = 0;              // set while enqueuing z = V(r) of a CG iteration whose level-0 UP kernel also forms r·z and beta
    int check_done = 0;          // set while enqueuing a solve cycle: kernels that can, return at once when scal->done
    int fused_grid = 0;          // CTAs of the last fused launch (= number of sum partials it wrote)
    int64_t launches = 0;
    char err[256] = "";
};

namespace {

int fail(wl_ctx* c, int code, const char* what, cudaError_t e = cudaSuccess) {
    if (c) {
        if (e != cudaSuccess) snprintf(c->err, sizeof(c->err), "%s: %s", what, cudaGetErrorString(e));
        else snprintf(c->err, sizeof(c->err), "%s", what);
    }
    return code;
}

#define CU(c, call)                                                      \
    do {                                                                 \
        cudaError_t e__ = (call);                                        \
        if (e__ != cudaSuccess) return fail((c), WL_ECUDA, #call, e__);  \
    } while (0)

#define KCHECK(c, name)                                                  \
    do {                                                                 \
        cudaError_t e__ = cudaGetLastError();                            \
        if (e__ != cudaSuccess) return fail((c), WL_ECUDA, name, e__);   \
        (c)->launches++;                                                 \
        (c)->pdl_armed = false;                                          \
    } while (0)

// Launch of a kernel that contains griddepcontrol.wait (fused level halves, coarse tail).  With WL_OPT_PDL it carries the
// programmatic-serialization attribute when the launch before it (same API call, same stream) was such a kernel too, so that
// the only things it reads before its wait — the level's coefficients and work plan — were written by an earlier, fully
// ordered launch.  A stream capture turns the attribute into a programmatic edge of the graph.
template <typename... KArgs, typename... Args>
cudaError_t launch_chained(wl_ctx* c, void (*kern)(KArgs...), int grid, int block, size_t smem, Args&&... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3((unsigned)block);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = c->stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = (c->opt_pdl && c->pdl_armed) ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, std::forward<Args>(args)...);
}
#define KCHAINED(c, name)                                                \
    do {                                                                 \
        KCHECK(c, name);                                                 \
        (c)->pdl_armed = true;                                           \
    } while (0)

inline int grid_for(const wl_ctx* c, long long work) {
    long long blocks = (work + kBlock - 1) / kBlock;
    long long cap = (long long)c->num_sms * 8;
    if (blocks < 1) blocks = 1;
    return (int)(blocks < cap ? blocks : cap);
}

inline int nparts_for(const wl_ctx* c, long long work) {
    int g = grid_for(c, work);
    return g < kMaxPartials ? g : kMaxPartials;
}

// ---- typed implementation ------------------------------------------------------------------------------------
template <typename T, int ND>
struct Impl {
    static T* P(void* p) { return (T*)p; }
    static const T* P(const void* p) { return (const T*)p; }

    // Row-wise 16-byte kernels need whole vectors per row and aligned arrays.
    static bool rows_ok(const Grid& g, const void* a, const void* b2 = nullptr, const void* c2 = nullptr) {
        constexpr int VEC = 16 / (int)sizeof(T);
        return g.N0 % VEC == 0 && (((uintptr_t)a | (uintptr_t)b2 | (uintptr_t)c2) & 15) == 0;
    }
    static int rows_grid(const wl_ctx* c, long long nrows) {
        long long blocks = (nrows + kRowsY - 1) / kRowsY;
        const long long cap = (long long)c->num_sms * 8;
        return (int)(blocks < 1 ? 1 : (blocks < cap ? blocks : cap));
    }

    static int set_coeff(wl_ctx* c, const void* Ldev) {
        Level& f = c->lev[0];
        if (rows_ok(f.g, Ldev, f.L)) {
            k_copy_coeff_rows<T, ND><<<rows_grid(c, (long long)f.g.N1 * f.g.N2 * ND), dim3(kRowsX, kRowsY), 0, c->stream>>>(f.g, P(Ldev), P(f.L));
            KCHECK(c, "k_copy_coeff_rows");
        } else {
            k_copy_coeff<T, ND><<<grid_for(c, f.g.M * ND), kBlock, 0, c->stream>>>(f.g, P(Ldev), P(f.L));
            KCHECK(c, "k_copy_coeff");
        }
        return finish_coeff(c);
    }

    // NEXT-3: level-0 coefficients from analytic bodies, evaluated on the device (wl_body.cuh), then the same chain.
    static int set_bodies(wl_ctx* c, int nbodies) {
        Level& f = c->lev[0];
        if (rows_ok(f.g, f.L)) {
            k_body_coeff_rows<T, ND><<<rows_grid(c, (long long)f.g.N1 * f.g.N2 * ND), dim3(kRowsX, kRowsY), 0, c->stream>>>(f.g, c->d_bodies, nbodies, P(f.L));
            KCHECK(c, "k_body_coeff_rows");
        } else {
            k_body_coeff<T, ND><<<grid_for(c, f.g.M * ND), kBlock, 0, c->stream>>>(f.g, c->d_bodies, nbodies, P(f.L));
            KCHECK(c, "k_body_coeff");
        }
        return finish_coeff(c);
    }

    // coarsening chain (one kernel per level, fixed summation tree) and omega/D per level
    static int finish_coeff(wl_ctx* c) {
        for (int l = 0; l + 1 < c->nlev; ++l) {
            Level& a = c->lev[l];
            Level& b = c->lev[l + 1];
            k_coarsen<T, ND><<<grid_for(c, b.g.M * ND), kBlock, 0, c->stream>>>(a.g, b.g, P(a.L), P(b.L));
            KCHECK(c, "k_coarsen");
        }
        for (int l = 0; USEC && ND == 3 && l < c->nlev; ++l) {   // omega·(1/D) per cell for the kernels that load it (fp64, 3-D)
            Level& v = c->lev[l];
            if (!v.C) continue;
            if (rows_ok(v.g, v.L, v.C)) {
                k_make_c_rows<T, ND><<<rows_grid(c, (long long)v.g.N1 * v.g.N2), dim3(kRowsX, kRowsY), 0, c->stream>>>(v.g, P(v.L), P(v.C));
                KCHECK(c, "k_make_c_rows");
            } else {
                k_make_c<T, ND><<<grid_for(c, v.g.M), kBlock, 0, c->stream>>>(v.g, P(v.L), P(v.C));
                KCHECK(c, "k_make_c");
            }
        }
        c->have_coeff = true;
        return WL_OK;
    }

    static int jacobi_sweep(wl_ctx* c, int l, const void* xin, const void* b, void* xout) {
        Level& v = c->lev[l];
        k_jacobi<T, ND><<<grid_for(c, v.g.M), kBlock, 0, c->stream>>>(v.g, P(v.L), P(xin), P(b), P(xout));
        KCHECK(c, "k_jacobi");
        return WL_OK;
    }

    // `sweeps` sweeps in place on x using `tmp` as the other half of the ping-pong; result always lands in x.
    static int jacobi(wl_ctx* c, int l, void* x, const void* b, void* tmp, int sweeps) {
        void* cur = x;
        void* oth = tmp;
        for (int s = 0; s < sweeps; ++s) {
            int rc = jacobi_sweep(c, l, cur, b, oth);
            if (rc) return rc;
            void* t = cur; cur = oth; oth = t;
        }
        if (cur != x) CU(c, cudaMemcpyAsync(x, cur, (size_t)c->lev[l].g.M * sizeof(T), cudaMemcpyDeviceToDevice, c->stream));
        return WL_OK;
    }

    static int residual_restrict(wl_ctx* c, int l, const void* x, const void* b, void* bc, void* xc) {
        Level& f = c->lev[l];
        Level& k = c->lev[l + 1];
        k_residual_restrict<T, ND><<<grid_for(c, k.g.M), kBlock, 0, c->stream>>>(f.g, k.g, P(f.L), P(x), P(b), P(bc), P(xc));
        KCHECK(c, "k_residual_restrict");
        return WL_OK;
    }

    static int prolong(wl_ctx* c, int l, const void* xc, void* x) {
        Level& f = c->lev[l];
        Level& k = c->lev[l + 1];
        k_prolong_add<T, ND><<<grid_for(c, f.g.M), kBlock, 0, c->stream>>>(f.g, k.g, P(xc), P(x));
        KCHECK(c, "k_prolong_add");
        return WL_OK;
    }

    static int ensure_tmp(wl_ctx* c, int l) {
        Level& v = c->lev[l];
        if (!v.tmp && cudaMalloc(&v.tmp, (size_t)v.g.M * sizeof(T)) != cudaSuccess) {
            cudaGetLastError();
            return fail(c, WL_ENOMEM, "cudaMalloc(level tmp)");
        }
        return WL_OK;
    }

    // DOWN half of level l with generic kernels: x_out = J(J(x_in)) (x_in == nullptr: from zero), bc = R(b - A x_out).
    static int down_generic(wl_ctx* c, int l, const void* x_in, const void* b, void* x_out, void* bc) {
        int rc;
        Level& v = c->lev[l];
        if ((rc = ensure_tmp(c, l))) return rc;
        if (x_in) {
            if ((rc = jacobi_sweep(c, l, x_in, b, v.tmp))) return rc;
        } else {
            k_jacobi_from_zero<T, ND><<<grid_for(c, v.g.M), kBlock, 0, c->stream>>>(v.g, P(v.L), P(b), P(v.tmp));
            KCHECK(c, "k_jacobi_from_zero");
        }
        if ((rc = jacobi_sweep(c, l, v.tmp, b, x_out))) return rc;
        return residual_restrict(c, l, x_out, b, bc, nullptr);
    }

    // UP half of level l with generic kernels: x_out = J(J(x_in + P xc)).
    static int up_generic(wl_ctx* c, int l, const void* x_in, const void* xc, const void* b, void* x_out) {
        int rc;
        Level& f = c->lev[l];
        Level& k = c->lev[l + 1];
        if ((rc = ensure_tmp(c, l))) return rc;
        k_prolong_out<T, ND><<<grid_for(c, f.g.M), kBlock, 0, c->stream>>>(f.g, k.g, P(xc), P(x_in), P(x_out));
        KCHECK(c, "k_prolong_out");
        if ((rc = jacobi_sweep(c, l, x_out, b, f.tmp))) return rc;
        return jacobi_sweep(c, l, f.tmp, b, x_out);
    }


    // ---- fused level halves (wl_fused3d.cuh) ---------------------------------------------------------------------
    // Tile and planes in flight (what fits 227 KB beside the exchange planes).  fp32: 64x16 cells, omega/D recomputed in
    // the kernel (5 planes per ring slot); fp64: 32x14 cells, omega/D read as a sixth plane (an IEEE fp64 division is ~20
    // instructions).  12 warps each.  Measured alternatives: profiles/r2_fused_ncu.md.
    static constexpr int FTX = sizeof(T) == 4 ? 64 : 32, FTY = sizeof(T) == 4 ? 16 : 14;
    static constexpr bool USEC = sizeof(T) == 8 && WL_FP64_C_PLANE != 0;
    template <bool PROLONG> static constexpr int FPF = (PROLONG && USEC) ? 2 : 3;   // fp32 DOWN with 4 planes in flight: no gain

    // Fused kernels apply to 3-D levels that have a coarser level, whose rows (and the coarse rows) are whole 16-byte
    // vectors; opt_fused == 1 keeps levels smaller than one tile on the generic kernels, 2 forces them (tests).
    static constexpr int F2TX = sizeof(T) == 4 ? 64 : 32, F2TY = 32;   // 2-D tile

    static bool fused_ok(const wl_ctx* c, int l) {
        if (!c->opt_fused || l + 1 >= c->nlev) return false;
        if (c->unaligned && l == c->unaligned_level) return false;   // TMA needs 16-byte aligned arrays: generic kernels instead
        const Grid& g = c->lev[l].g;
        constexpr int VEC = 16 / (int)sizeof(T);
        if (g.N0 % (2 * VEC)) return false;
        if (ND == 3) {
            if (c->opt_fused == 1 && (g.N0 < FTX / 2 || g.N1 < 16 || g.N2 < 8)) return false;
        } else {
            if (c->opt_fused == 1 && (g.N0 < F2TX / 2 || g.N1 < F2TY / 2)) return false;
            const long long tiles = (long long)((g.N0 + F2TX - 1) / F2TX) * ((g.N1 + F2TY - 1) / F2TY);
            if (tiles > kMaxPartials) return false;
        }
        return get_encode_tiled() != nullptr;
    }

    static bool map_cells2(CUtensorMap* m, const void* base, const Grid& g, bool coarse_box) {
        using G = F2<T, F2TX, F2TY>;
        if (((uintptr_t)base & 15) != 0) return false;
        const uint64_t d[3] = {(uint64_t)g.N0, (uint64_t)g.N1, 1};
        const uint32_t b[3] = {(uint32_t)(coarse_box ? G::CWX : G::WX), (uint32_t)(coarse_box ? G::CWY : G::WY), 1u};
        return encode_map(m, base, (int)sizeof(T), 2, d, b);
    }

    template <bool PROLONG, bool ZERO_IN, bool SHIFT, bool STAGE3, bool RESTRICT, bool NORMS, bool RIN = false, bool TICKET = false>
    static int launch_fused2(wl_ctx* c, int l, const void* x_in, const void* xc, const void* b, void* x_out, void* bc) {
        using G = F2<T, F2TX, F2TY>;
        Level& f = c->lev[l];
        CUtensorMap mx, mb, mL0, mL1, mxc;
        bool ok = map_cells2(&mb, b, f.g, false) && map_cells2(&mL0, P(f.L), f.g, false) && map_cells2(&mL1, P(f.L) + f.g.M, f.g, false);
        if (ZERO_IN) mx = mb; else ok = ok && map_cells2(&mx, x_in, f.g, false);
        if (PROLONG) ok = ok && map_cells2(&mxc, xc, c->lev[l + 1].g, true); else mxc = mb;
        if (!ok) return fail(c, WL_ECUDA, "cuTensorMapEncodeTiled refused a level array (alignment?)");
        Fused2Params<T> prm;
        prm.N0 = f.g.N0; prm.N1 = f.g.N1;
        prm.tiles_x = (f.g.N0 + F2TX - 1) / F2TX;
        prm.tiles_y = (f.g.N1 + F2TY - 1) / F2TY;
        prm.xout = P(x_out);
        prm.bc = P(bc);
        prm.scal = c->d_scal;
        prm.partials = c->d_partials;
        prm.hist = c->d_hist;
        prm.host_scal = c->h_scal;
        prm.host_hist = c->h_hist;
        prm.cells = f.g.M;
        prm.check_done = c->check_done;
        const int grid = prm.tiles_x * prm.tiles_y;
        c->fused_grid = grid;
        launch_chained(c, k_fused2d<T, F2TX, F2TY, PROLONG, ZERO_IN, SHIFT, STAGE3, RESTRICT, NORMS, RIN, TICKET>, grid, G::NT,
                       fused2d_smem_bytes<T, F2TX, F2TY>(), mx, mb, mL0, mL1, mxc, prm);
        KCHAINED(c, "k_fused2d");
        return WL_OK;
    }

    static bool map_cells(CUtensorMap* m, const void* base, const Grid& g, bool coarse_box) {
        using G = F3<T, FTX, FTY>;
        if (((uintptr_t)base & 15) != 0) return false;
        const uint64_t d[3] = {(uint64_t)g.N0, (uint64_t)g.N1, (uint64_t)g.N2};
        const uint32_t b[3] = {(uint32_t)(coarse_box ? G::CWX : G::WX), (uint32_t)(coarse_box ? G::CWY : G::WY), 1u};
        return encode_map(m, base, (int)sizeof(T), 3, d, b);
    }

    template <bool PROLONG, bool ZERO_IN, bool SHIFT, bool STAGE3, bool RESTRICT, bool NORMS, bool RIN = false, bool TICKET = false>
    static int launch_fused(wl_ctx* c, int l, const void* x_in, const void* xc, const void* b, void* x_out, void* bc) {
        if constexpr (ND == 3) {
            using G = F3<T, FTX, FTY>;
            Level& f = c->lev[l];
            CUtensorMap mx, mb, mL0, mL1, mL2, mC, mxc;
            bool ok = map_cells(&mb, b, f.g, false);
            ok = ok && map_cells(&mL0, P(f.L), f.g, false) && map_cells(&mL1, P(f.L) + f.g.M, f.g, false) &&
                 map_cells(&mL2, P(f.L) + 2 * f.g.M, f.g, false);
            if (USEC) ok = ok && map_cells(&mC, P(f.C), f.g, false); else mC = mb;
            if (ZERO_IN) mx = mb; else ok = ok && map_cells(&mx, x_in, f.g, false);
            if (PROLONG) ok = ok && map_cells(&mxc, xc, c->lev[l + 1].g, true); else mxc = mb;
            if (!ok) return fail(c, WL_ECUDA, "cuTensorMapEncodeTiled refused a level array (alignment?)");
            Fused3Params<T> prm;
            prm.N0 = f.g.N0; prm.N1 = f.g.N1; prm.N2 = f.g.N2;
            if (!f.plan_items) return fail(c, WL_ECUDA, "fused level without a work plan");
            prm.items = f.plan_items;
            prm.item_start = f.plan_start;
            prm.xout = P(x_out);
            prm.bc = P(bc);
            prm.scal = c->d_scal;
            prm.partials = c->d_partials;
            prm.hist = c->d_hist;
            prm.host_scal = c->h_scal;
            prm.host_hist = c->h_hist;
            prm.cells = f.g.M;
            prm.negzero2 = 0x8000000080000000ULL;
            prm.check_done = c->check_done;
            prm.pcg = (NORMS && c->pcg_up) ? 1 : 0;
            auto kern = k_fused3d<T, FTX, FTY, FPF<PROLONG>, PROLONG, ZERO_IN, SHIFT, STAGE3, RESTRICT, NORMS, RIN, USEC, TICKET>;
            constexpr size_t smem = fused3d_smem_bytes<T, FTX, FTY, FPF<PROLONG>, PROLONG, USEC>();
            const int g = f.plan_grid;
            c->fused_grid = g;
            launch_chained(c, kern, g, G::NT, smem, mx, mb, mL0, mL1, mL2, mC, mxc, prm);
            KCHAINED(c, "k_fused3d");
            return WL_OK;
        } else {
            return launch_fused2<PROLONG, ZERO_IN, SHIFT, STAGE3, RESTRICT, NORMS, RIN, TICKET>(c, l, x_in, xc, b, x_out, bc);
        }
    }

    // DOWN half of level l: x_out = J(J(x_in)) (x_in == nullptr: from zero), bc = R(b - A x_out).
    static int down(wl_ctx* c, int l, const void* x_in, const void* b, void* x_out, void* bc) {
        if (!fused_ok(c, l)) return down_generic(c, l, x_in, b, x_out, bc);
        if (c->solve_kernels_now && l == 0 && x_in && c->d_hist)   // the instance wl_solve's graph launches (profiling / bench)
            return launch_fused<false, false, true, true, true, false, true, true>(c, l, x_in, nullptr, b, x_out, bc);
        if (x_in) return launch_fused<false, false, false, true, true, false>(c, l, x_in, nullptr, b, x_out, bc);
        return launch_fused<false, true, false, true, true, false>(c, l, nullptr, nullptr, b, x_out, bc);
    }

    // UP half of level l: x_out = J(J(x_in + P xc)).
    static int up(wl_ctx* c, int l, const void* x_in, const void* xc, const void* b, void* x_out) {
        if (!fused_ok(c, l)) return up_generic(c, l, x_in, xc, b, x_out);
        if ((c->solve_kernels_now || c->pcg_up) && l == 0 && c->d_hist)
            return launch_fused<true, false, false, false, false, true, false, true>(c, l, x_in, xc, b, x_out, nullptr);
        return launch_fused<true, false, false, false, false, false>(c, l, x_in, xc, b, x_out, nullptr);
    }

    // VCYCLE(l) for a level inside the coarse tail: one persistent CTA (wl_tail.cuh).  x_in == nullptr: zero guess.
    static int tail(wl_ctx* c, int l, const void* x_in, const void* b, void* x_out) {
        TailParams<T> prm;
        prm.nl = c->nlev - l;
        prm.zero_in = x_in ? 0 : 1;
        prm.coarsest_is_correction = (c->nlev > 1) ? 1 : 0;
        unsigned off = 0;
        for (int k = 0; k < prm.nl; ++k) {
            const Level& v = c->lev[l + k];
            prm.g[k] = v.g;
            prm.L[k] = P(v.L);
            prm.off[k] = off;
            off += (unsigned)(((size_t)(4 + ND) * v.g.M * sizeof(T) + 15) / 16 * 16);
        }
        prm.x_in = P(x_in);
        prm.b_in = P(b);
        prm.x_out = P(x_out);
        prm.scal = c->d_scal;
        prm.check_done = c->check_done;
        auto kern = k_coarse_tail<T, ND>;
        launch_chained(c, kern, 1, kTailThreads, off, prm);
        KCHAINED(c, "k_coarse_tail");
        return WL_OK;
    }

    // 64 sweeps on the coarsest level.  x_in == nullptr: from zero (correction level), result in x_out; the other
    // buffer `x_mid` is the second half of the ping-pong.  x_in != nullptr (a one-level hierarchy): x_in may be x_out.
    static int coarsest(wl_ctx* c, int l, const void* x_in, const void* b, void* x_mid, void* x_out) {
        Level& v = c->lev[l];
        int rc;
        if (!x_in) {
            k_jacobi_from_zero<T, ND><<<grid_for(c, v.g.M), kBlock, 0, c->stream>>>(v.g, P(v.L), P(b), P(x_mid));
            KCHECK(c, "k_jacobi_from_zero");
            void* cur = x_mid;
            void* oth = x_out;
            for (int s = 1; s < 64; ++s) {  // 63 more: x_mid -> x_out -> ... -> x_out
                if ((rc = jacobi_sweep(c, l, cur, b, oth))) return rc;
                void* t2 = cur; cur = oth; oth = t2;
            }
            return WL_OK;
        }
        if (x_in != x_out) CU(c, cudaMemcpyAsync(x_out, x_in, (size_t)v.g.M * sizeof(T), cudaMemcpyDeviceToDevice, c->stream));
        return jacobi(c, l, x_out, b, x_mid, 64);
    }

    // VCYCLE(l): x_out = cycle(x_in) on level l; x_mid = level-sized scratch (may not alias x_in / x_out).
    // x_in == nullptr means a zero initial guess (every correction level).
    static int vcycle(wl_ctx* c, int l, const void* x_in, const void* b, void* x_mid, void* x_out) {
        int rc;
        if (c->opt_coarse_cta && l >= c->tail_first)
            return tail(c, l, (l == c->nlev - 1 && l > 0) ? nullptr : x_in, b, x_out);
        if (l == c->nlev - 1) return coarsest(c, l, (c->nlev > 1 && l > 0) ? nullptr : x_in, b, x_mid, x_out);
        Level& k = c->lev[l + 1];
        if ((rc = down(c, l, x_in, b, x_mid, k.b))) return rc;
        if ((rc = vcycle(c, l + 1, nullptr, k.b, k.x[0], k.x[1]))) return rc;
        return up(c, l, x_mid, k.x[1], b, x_out);
    }

    // Σp -> mean (ordered), p -= mean.
    static int remove_mean(wl_ctx* c, void* p) {
        const long long M = c->lev[0].g.M;
        const int np = nparts_for(c, M);
        k_sum<T><<<np, kBlock, 0, c->stream>>>(M, P(p), c->d_partials);
        KCHECK(c, "k_sum");
        k_finish_mean<<<1, 32, 0, c->stream>>>(c->d_scal, c->d_partials, np, M);
        KCHECK(c, "k_finish_mean");
        k_shift<T><<<grid_for(c, M), kBlock, 0, c->stream>>>(M, P(p), c->d_scal);
        KCHECK(c, "k_shift");
        return WL_OK;
    }

    // ||b - A p||inf into slot 1 (and Σp partials -> mean, not applied).
    static int resnorm(wl_ctx* c, const void* p, const void* b) {
        Level& f = c->lev[0];
        const int np = nparts_for(c, f.g.M);
        k_zero_slot<<<1, 32, 0, c->stream>>>(c->d_scal, 1);
        KCHECK(c, "k_zero_slot");
        k_resnorm_sum<T, ND><<<np, kBlock, 0, c->stream>>>(f.g, P(f.L), P(p), P(b), c->d_scal, 1, c->d_partials);
        KCHECK(c, "k_resnorm_sum");
        k_finish_mean<<<1, 32, 0, c->stream>>>(c->d_scal, c->d_partials, np, f.g.M);
        KCHECK(c, "k_finish_mean");
        return WL_OK;
    }

    static int absmax_b(wl_ctx* c, const void* b) {
        const long long M = c->lev[0].g.M;
        k_zero_slot<<<1, 32, 0, c->stream>>>(c->d_scal, 0);
        KCHECK(c, "k_zero_slot");
        k_absmax<T><<<grid_for(c, M), kBlock, 0, c->stream>>>(M, P(b), c->d_scal, 0);
        KCHECK(c, "k_absmax");
        return WL_OK;
    }

    // The mean removal of cycle k can ride on cycle k+1: its level-0 DOWN kernel subtracts (T)mean from p on load (exactly
    // the value the oracle stores), the last cycle's shift is applied by one k_shift pass.  Needs the fused level 0.
    static bool can_defer(const wl_ctx* c) { return c->nlev > 1 && c->tail_first > 0 && fused_ok(c, 0); }

    // A cycle may be enqueued before the previous one's stop test is known only if every kernel of it that writes
    // the iterate checks scal->done: all levels above the tail fused, the rest in the tail CTA.
    static bool can_speculate(const wl_ctx* c) {
        if (!c->opt_coarse_cta || c->tail_first >= c->nlev || c->tail_first == 0) return false;
        for (int l = 0; l < c->tail_first; ++l)
            if (!fused_ok(c, l)) return false;
        return true;
    }

    // Generic-path scratch is allocated before a stream capture starts.
    static int prepare(wl_ctx* c) {
        for (int l = 0; l + 1 < c->nlev && l < (c->opt_coarse_cta ? c->tail_first : c->nlev); ++l)
            if (!fused_ok(c, l)) { int rc = ensure_tmp(c, l); if (rc) return rc; }
        if (!(c->opt_coarse_cta && c->tail_first < c->nlev)) { /* coarsest level runs on the generic kernels */ }
        return WL_OK;
    }

    // One V-cycle in the oracle's literal order: VCYCLE(0), p -= mean(p), ||b - A p||inf of the shifted p (slot 1).
    // Used by wl_vcycle and by solves whose level 0 is not fused; the fused solve uses cycle_lagged.
    static int cycle(wl_ctx* c, void* p, const void* b) {
        int rc;
        if ((rc = vcycle(c, 0, p, b, c->lev[0].x[1], p))) return rc;
        if ((rc = remove_mean(c, p))) return rc;
        return resnorm(c, p, b);
    }

    static int apply_shift(wl_ctx* c, void* p) {
        const long long M = c->lev[0].g.M;
        k_shift<T><<<grid_for(c, M), kBlock, 0, c->stream>>>(M, P(p), c->d_scal);
        KCHECK(c, "k_shift");
        return WL_OK;
    }

    // The solve cycle with the lagged stop test: DOWN0 measures the residual of its input for free and its
    // last CTA records it and takes the stop decision; UP0 needs no residual stage (2 stencil stages instead of 3), only
    // sums p, and its last CTA finishes the mean and bumps the cycle counter.  No single-thread kernels in the cycle.
    static int cycle_lagged(wl_ctx* c, void* p, const void* b) {
        int rc;
        Level& k1 = c->lev[1];
        if ((rc = launch_fused<false, false, true, true, true, false, true, true>(c, 0, p, nullptr, b, c->lev[0].x[1], k1.b))) return rc;
        if ((rc = vcycle(c, 1, nullptr, k1.b, k1.x[0], k1.x[1]))) return rc;
        return launch_fused<true, false, false, false, false, true, false, true>(c, 0, c->lev[0].x[1], k1.x[1], b, p, nullptr);
    }

    // ---- V-cycle-preconditioned conjugate gradients (wl_pcg.cuh) ------------------------------------
    static int pcg_residual(wl_ctx* c, const void* x, const void* b) {
        Level& f = c->lev[0];
        if (rows_ok(f.g, f.L, x, b)) {
            const int gr = rows_grid(c, (long long)f.g.N1 * f.g.N2);
            k_pcg_Ap_rows<T, ND, true><<<gr, dim3(kRowsX, kRowsY), 0, c->stream>>>(f.g, P(f.L), P(x), P(c->cg_v[0]), c->d_scal, c->d_partials, P(b),
                                                                                  c->d_hist, c->h_scal, c->h_hist);
            KCHECK(c, "k_pcg_Ap_rows");
            return WL_OK;
        }
        k_pcg_residual<T, ND><<<nparts_for(c, f.g.M), kBlock, 0, c->stream>>>(f.g, P(f.L), P(x), P(b), P(c->cg_v[0]), c->d_scal, c->d_hist,
                                                                           c->h_scal, c->h_hist);
        KCHECK(c, "k_pcg_residual");
        return WL_OK;
    }
    // one iteration: z = V(r); rho', beta; p; q = A p, alpha; x, r, hist
    static int pcg_iteration(wl_ctx* c, void* x) {
        Level& f = c->lev[0];
        const long long M = f.g.M;
        T* r = P(c->cg_v[0]); T* z = P(c->cg_v[1]); T* p = P(c->cg_v[2]); T* q = P(c->cg_v[3]);
        int rc;
        // with a fused 3-D level 0 the last kernel of the V-cycle (level-0 UP) also forms sum z, sum r z and beta
        const bool dot_in_up = ND == 3 && c->nlev > 1 && c->tail_first > 0 && fused_ok(c, 0) && c->d_hist;
        c->pcg_up = dot_in_up ? 1 : 0;
        rc = vcycle(c, 0, nullptr, r, f.x[1], z);
        c->pcg_up = 0;
        if (rc) return rc;
        const int np = nparts_for(c, M) < kMaxPartials / 2 ? nparts_for(c, M) : kMaxPartials / 2;
        if (!dot_in_up) {
            k_pcg_dot_rz<T><<<np, kBlock, 0, c->stream>>>(M, r, z, c->d_scal, c->d_partials);
            KCHECK(c, "k_pcg_dot_rz");
        }
        const bool vec = rows_ok(f.g, x, nullptr, nullptr);   // the work vectors are the context's own (aligned); x is the caller's
        if (vec) {
            k_pcg_update_p_vec<T><<<grid_for(c, M / (16 / (long long)sizeof(T))), kBlock, 0, c->stream>>>(M, z, p, c->d_scal);
            KCHECK(c, "k_pcg_update_p_vec");
        } else {
            k_pcg_update_p<T><<<grid_for(c, M), kBlock, 0, c->stream>>>(M, z, p, c->d_scal);
            KCHECK(c, "k_pcg_update_p");
        }
        if (rows_ok(f.g, f.L, p, q)) {
            const int gr = rows_grid(c, (long long)f.g.N1 * f.g.N2);
            k_pcg_Ap_rows<T, ND, false><<<gr < kMaxPartials ? gr : kMaxPartials, dim3(kRowsX, kRowsY), 0, c->stream>>>(f.g, P(f.L), p, q, c->d_scal, c->d_partials, nullptr, nullptr, nullptr, nullptr);
            KCHECK(c, "k_pcg_Ap_rows");
        } else {
            k_pcg_Ap<T, ND><<<np, kBlock, 0, c->stream>>>(f.g, P(f.L), p, q, c->d_scal, c->d_partials);
            KCHECK(c, "k_pcg_Ap");
        }
        if (vec) k_pcg_update_xr<T, true><<<np, kBlock, 0, c->stream>>>(M, P(x), r, p, q, c->d_scal, c->d_hist, c->h_scal, c->h_hist);
        else k_pcg_update_xr<T, false><<<np, kBlock, 0, c->stream>>>(M, P(x), r, p, q, c->d_scal, c->d_hist, c->h_scal, c->h_hist);
        KCHECK(c, "k_pcg_update_xr");
        return WL_OK;
    }

    // Set every opt-in shared-memory size once, outside any stream capture.
    static int init_kernels(wl_ctx* c) {
        if constexpr (ND == 3) {
            // work plans of the fused level halves (every level that has a coarser one; tiny levels included: WL_OPT_FUSED = 2)
            for (int l = 0; l + 1 < c->nlev; ++l) {
                Level& v = c->lev[l];
                const Plan pl = plan_fused3d(v.g.N0, v.g.N1, v.g.N2, FTX, FTY, c->num_sms);
                static_assert(sizeof(PlanItem) == sizeof(int4), "plan items are uploaded as int4");
                if (cudaMalloc((void**)&v.plan_items, pl.items.size() * sizeof(int4)) != cudaSuccess ||
                    cudaMalloc((void**)&v.plan_start, pl.start.size() * sizeof(int)) != cudaSuccess)
                    return fail(c, WL_ENOMEM, "cudaMalloc(work plan)");
                CU(c, cudaMemcpy(v.plan_items, pl.items.data(), pl.items.size() * sizeof(int4), cudaMemcpyHostToDevice));
                CU(c, cudaMemcpy(v.plan_start, pl.start.data(), pl.start.size() * sizeof(int), cudaMemcpyHostToDevice));
                v.plan_grid = pl.grid();
            }
            constexpr int s0 = (int)fused3d_smem_bytes<T, FTX, FTY, FPF<false>, false, USEC>(), s1 = (int)fused3d_smem_bytes<T, FTX, FTY, FPF<true>, true, USEC>();
            constexpr auto A = cudaFuncAttributeMaxDynamicSharedMemorySize;
            CU(c, cudaFuncSetAttribute(k_fused3d<T, FTX, FTY, FPF<false>, false, false, false, true, true, false, false, USEC, false>, A, s0));
            CU(c, cudaFuncSetAttribute(k_fused3d<T, FTX, FTY, FPF<false>, false, true, false, true, true, false, false, USEC, false>, A, s0));
            CU(c, cudaFuncSetAttribute(k_fused3d<T, FTX, FTY, FPF<true>, true, false, false, false, false, false, false, USEC, false>, A, s1));
            CU(c, cudaFuncSetAttribute(k_fused3d<T, FTX, FTY, FPF<false>, false, false, true, true, true, false, true, USEC, true>, A, s0));
            CU(c, cudaFuncSetAttribute(k_fused3d<T, FTX, FTY, FPF<true>, true, false, false, false, false, true, false, USEC, true>, A, s1));
        }
        if constexpr (ND == 2) {
            constexpr int s2 = (int)fused2d_smem_bytes<T, F2TX, F2TY>();
            constexpr auto A = cudaFuncAttributeMaxDynamicSharedMemorySize;
            CU(c, cudaFuncSetAttribute(k_fused2d<T, F2TX, F2TY, false, false, false, true, true, false, false, false>, A, s2));
            CU(c, cudaFuncSetAttribute(k_fused2d<T, F2TX, F2TY, false, true, false, true, true, false, false, false>, A, s2));
            CU(c, cudaFuncSetAttribute(k_fused2d<T, F2TX, F2TY, true, false, false, false, false, false, false, false>, A, s2));
            CU(c, cudaFuncSetAttribute(k_fused2d<T, F2TX, F2TY, false, false, true, true, true, false, true, true>, A, s2));
            CU(c, cudaFuncSetAttribute(k_fused2d<T, F2TX, F2TY, true, false, false, false, false, true, false, true>, A, s2));
        }
        CU(c, cudaFuncSetAttribute(k_coarse_tail<T, ND>, cudaFuncAttributeMaxDynamicSharedMemorySize, kTailSmemBudget));
        if constexpr (ND == 3)
            CU(c, cudaFuncSetAttribute(k_convdiff3d<T, CDTY>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)CD3<T, CDTY>::smem_bytes()));
        return WL_OK;
    }

    // NEXT-4: r = convdiff(u; nu).  Tiled TMA kernel for 3-D grids whose rows are whole 16-byte vectors, else one thread per cell.
    // rows per tile: fp32 11 + the flux-only row = 12 warps, three per scheduler (measured 512^3: 2.69 ms; 8 rows: 2.96 ms);
    // fp64 8 (256^3: 1.03 ms; 11 rows: 1.19 ms)
    static constexpr int CDTY = sizeof(T) == 4 ? 11 : 8;
    static int convdiff(wl_ctx* c, const void* u, double nu, void* r) {
        const Grid& g = c->lev[0].g;
        if constexpr (ND == 3) {
            using G = CD3<T, CDTY>;
            if (c->opt_fused != 0 && rows_ok(g, u, r)) {
                CUtensorMap m[3];
                const uint64_t d[3] = {(uint64_t)g.N0, (uint64_t)g.N1, (uint64_t)g.N2};
                const uint32_t bx[3] = {(uint32_t)G::WX, (uint32_t)G::WY, 1u};
                bool ok = true;
                for (int i = 0; i < 3; ++i) ok = ok && encode_map(&m[i], P(u) + (long long)i * g.M, (int)sizeof(T), 3, d, bx);
                if (!ok) return fail(c, WL_ECUDA, "cuTensorMapEncodeTiled refused the velocity field");
                CdParams<T> prm;
                prm.N0 = g.N0; prm.N1 = g.N1; prm.N2 = g.N2;
                prm.ntx = (g.N0 + G::TX - 1) / G::TX;
                prm.nty = (g.N1 + G::TY - 1) / G::TY;
                prm.nz = convdiff_chunk(prm.ntx * prm.nty, g.N2, c->num_sms * convdiff_ctas_per_sm());
                prm.nu = (T)nu;
                prm.r = P(r);
                prm.M = g.M;
                prm.negzero2 = 0x8000000080000000ULL;
                const int nchunks = (g.N2 + prm.nz - 1) / prm.nz;
                k_convdiff3d<T, CDTY><<<prm.ntx * prm.nty * nchunks, G::NT, G::smem_bytes(), c->stream>>>(m[0], m[1], m[2], prm);
                KCHECK(c, "k_convdiff3d");
                return WL_OK;
            }
        }
        k_convdiff<T, ND><<<grid_for(c, g.M), kBlock, 0, c->stream>>>(g, P(u), (T)nu, P(r));
        KCHECK(c, "k_convdiff");
        return WL_OK;
    }
    static int convdiff_ctas_per_sm() {
        const size_t b = CD3<T, CDTY>::smem_bytes() + 1024;
        const int by_smem = (int)((size_t)227 * 1024 / b);
        const int by_threads = 2048 / CD3<T, CDTY>::NT;
        const int k = by_smem < by_threads ? by_smem : by_threads;
        return k < 1 ? 1 : k;
    }
    // planes per z-chunk: the split of N2 that minimises waves x (planes + 1 extra flux step) over `slots` resident CTAs
    static int convdiff_chunk(int tiles, int N2, int slots) {
        int best = N2;
        long long best_cost = -1;
        for (int nch = 1; nch <= N2; ++nch) {
            const int nz = (N2 + nch - 1) / nch;
            const int real = (N2 + nz - 1) / nz;
            const long long items = (long long)tiles * real;
            const long long waves = (items + slots - 1) / slots;
            const long long cost = waves * (nz + 2);
            if (best_cost < 0 || cost < best_cost) { best_cost = cost; best = nz; }
            if (nz == 1) break;
        }
        return best;
    }

    // with_nb: also leave ||b||inf in slot 0 (fused into the row kernel; one more pass on the generic path)
    static int divergence(wl_ctx* c, const void* u, void* b, bool with_nb) {
        Level& f = c->lev[0];
        if (rows_ok(f.g, u, b)) {
            if (with_nb) {
                k_zero_slot<<<1, 32, 0, c->stream>>>(c->d_scal, 0);
                KCHECK(c, "k_zero_slot");
            }
            k_divergence_rows<T, ND><<<rows_grid(c, (long long)f.g.N1 * f.g.N2), dim3(kRowsX, kRowsY), 0, c->stream>>>(f.g, P(u), P(b), with_nb ? c->d_scal : nullptr);
            KCHECK(c, "k_divergence_rows");
            return WL_OK;
        }
        k_divergence<T, ND><<<grid_for(c, f.g.M), kBlock, 0, c->stream>>>(f.g, P(u), P(b));
        KCHECK(c, "k_divergence");
        return with_nb ? absmax_b(c, b) : WL_OK;
    }

    static int gradient(wl_ctx* c, void* u, const void* p) {
        Level& f = c->lev[0];
        if (rows_ok(f.g, u, p, f.L)) {
            k_gradient_rows<T, ND><<<rows_grid(c, (long long)f.g.N1 * f.g.N2), dim3(kRowsX, kRowsY), 0, c->stream>>>(f.g, P(f.L), P(u), P(p));
            KCHECK(c, "k_gradient_rows");
            return WL_OK;
        }
        k_gradient<T, ND><<<grid_for(c, f.g.M), kBlock, 0, c->stream>>>(f.g, P(f.L), P(u), P(p));
        KCHECK(c, "k_gradient");
        return WL_OK;
    }
};

#define DISPATCH(c, call)                                                         \
    ((c)->dtype == WL_F32 ? ((c)->n == 2 ? Impl<float, 2>::call : Impl<float, 3>::call) \
                          : ((c)->n == 2 ? Impl<double, 2>::call : Impl<double, 3>::call))

int read_scalars(wl_ctx* c) {
    CU(c, cudaMemcpyAsync(c->h_scal, c->d_scal, sizeof(Scalars), cudaMemcpyDeviceToHost, c->stream));
    CU(c, cudaStreamSynchronize(c->stream));
    return WL_OK;
}

inline double bits_to_double(unsigned long long b) {
    double d;
    memcpy(&d, &b, sizeof(d));
    return d;
}

void drop_graph(wl_ctx* c);

int ensure_hist(wl_ctx* c, int maxcycles) {
    if (maxcycles + 1 <= c->hist_cap) return WL_OK;
    drop_graph(c);   // the cached graph holds the old history pointers
    if (c->d_hist) cudaFree(c->d_hist);
    if (c->h_hist) cudaFreeHost(c->h_hist);
    c->d_hist = nullptr; c->h_hist = nullptr; c->hist_cap = 0;
    int cap = maxcycles + 1 < 64 ? 64 : maxcycles + 1;
    if (cudaMalloc(&c->d_hist, sizeof(double) * cap) != cudaSuccess) return fail(c, WL_ENOMEM, "cudaMalloc(hist)");
    if (cudaMallocHost(&c->h_hist, sizeof(double) * cap) != cudaSuccess) return fail(c, WL_ENOMEM, "cudaMallocHost(hist)");
    c->hist_cap = cap;
    return WL_OK;
}

void drop_graph(wl_ctx* c) {
    for (auto& e : c->cg) {
        if (e.exec) cudaGraphExecDestroy(e.exec);
        e = wl_ctx::GraphEntry();
    }
}

// One V-cycle (+ k_cycle_end bookkeeping when `in_solve`) on the ctx stream: a cached CUDA graph when WL_OPT_GRAPH is on.
// variant: bit 0 = in_solve, bit 1 = lagged, 4 = one conjugate-gradient iteration (p = the iterate x, b unused).
int run_cycle(wl_ctx* c, void* p, const void* b, bool in_solve, bool lagged, bool pcg = false) {
    int rc;
    const int variant = pcg ? 4 : ((in_solve ? 1 : 0) | (lagged ? 2 : 0));
    auto enqueue = [&]() -> int {
        c->pdl_armed = false;   // the first kernel of a cycle is fully ordered after whatever precedes it in the stream
        c->check_done = in_solve ? 1 : 0;
        int r = pcg ? DISPATCH(c, pcg_iteration)(c, p) : (lagged ? DISPATCH(c, cycle_lagged)(c, p, b) : DISPATCH(c, cycle)(c, p, b));
        c->check_done = 0;
        if (r) return r;
        if (in_solve && !lagged && !pcg) {
            k_cycle_end<<<1, 32, 0, c->stream>>>(c->d_scal, c->d_hist, 0, c->h_scal, c->h_hist);
            KCHECK(c, "k_cycle_end");
        }
        return WL_OK;
    };
    if (!c->opt_graph) return enqueue();
    cudaStream_t user = c->stream;
    const bool proxy = (user == nullptr || user == cudaStreamLegacy || user == cudaStreamPerThread);
    cudaStream_t gs = proxy ? c->own_stream : user;
    wl_ctx::GraphEntry* ge = nullptr;
    for (auto& e : c->cg)
        if (e.exec && e.p == p && e.b == b && e.variant == variant) ge = &e;
    if (!ge) {
        ge = &c->cg[0];
        for (auto& e : c->cg)                       // a free entry, else the least recently used one
            if (!e.exec || (ge->exec && e.stamp < ge->stamp)) { ge = &e; if (!e.exec) break; }
        if (ge->exec) cudaGraphExecDestroy(ge->exec);
        *ge = wl_ctx::GraphEntry();
        if ((rc = DISPATCH(c, prepare)(c))) return rc;
        const int64_t before = c->launches;
        CU(c, cudaStreamBeginCapture(gs, cudaStreamCaptureModeThreadLocal));
        c->stream = gs;
        rc = enqueue();
        c->stream = user;
        cudaGraph_t graph = nullptr;
        cudaError_t e = cudaStreamEndCapture(gs, &graph);
        ge->nodes = c->launches - before;
        c->launches = before;
        if (rc) { if (graph) cudaGraphDestroy(graph); return rc; }
        if (e != cudaSuccess) return fail(c, WL_ECUDA, "cudaStreamEndCapture", e);
        e = cudaGraphInstantiate(&ge->exec, graph, 0);
        cudaGraphDestroy(graph);
        if (e != cudaSuccess) { ge->exec = nullptr; return fail(c, WL_ECUDA, "cudaGraphInstantiate", e); }
        ge->p = p; ge->b = b; ge->variant = variant;
    }
    ge->stamp = ++c->cg_clock;
    if (proxy) {
        CU(c, cudaEventRecord(c->ev_in, user));
        CU(c, cudaStreamWaitEvent(gs, c->ev_in, 0));
    }
    CU(c, cudaGraphLaunch(ge->exec, gs));
    if (proxy) {
        CU(c, cudaEventRecord(c->ev_out, gs));
        CU(c, cudaStreamWaitEvent(user, c->ev_out, 0));
    }
    c->launches += ge->nodes;
    return WL_OK;
}

// Spin on the pinned mirror until cycle `target` has been recorded by k_cycle_end; checks the stream now and then so a
// faulted or drained stream cannot hang the host.
int wait_cycle(wl_ctx* c, int target) {
    volatile Scalars* hm = c->h_scal;
    cudaStream_t user = c->stream;
    const bool proxy = c->opt_graph && (user == nullptr || user == cudaStreamLegacy || user == cudaStreamPerThread);
    cudaStream_t gs = proxy ? c->own_stream : user;
    for (unsigned spins = 0;; ++spins) {
        if (hm->cycle >= target) return WL_OK;
#if defined(__x86_64__) || defined(__i386__)
        __builtin_ia32_pause();
#endif
        if ((spins & 0xfff) == 0xfff) {
            cudaError_t e = cudaStreamQuery(gs);
            if (e == cudaSuccess && gs != user) e = cudaStreamQuery(user);
            if (e == cudaSuccess) {
                if (hm->cycle >= target) return WL_OK;
                return fail(c, WL_ECUDA, "wl_solve: the stream drained without recording the cycle");
            }
            if (e != cudaErrorNotReady) return fail(c, WL_ECUDA, "wl_solve: cudaStreamQuery", e);
        }
    }
}

// have_nb: ||b||inf is already in slot 0 (wl_project's divergence kernel left it there).
int solve_impl(wl_ctx* c, void* p, const void* b, double tol, int maxcycles, double* hist, int* ncycles, bool have_nb = false) {
    int rc;
    if ((rc = ensure_hist(c, maxcycles))) return rc;
    if (!have_nb && (rc = DISPATCH(c, absmax_b)(c, b))) return rc;
    const bool spec = DISPATCH(c, can_speculate)(c);
    const bool lagged = spec && DISPATCH(c, can_defer)(c);
    volatile Scalars* hm = c->h_scal;
    double nb = 0.0;
    int k = 0;
    if (lagged) {
        // Lagged stop test: launch g's level-0 DOWN kernel measures ||b - A p_{g-1}||inf (g = 1: the
        // initial residual) and k_cycle_check decides on the device; two launches stay enqueued, the host polls the
        // pinned mirror instead of synchronising, so the GPU never waits for a host round trip.
        CU(c, cudaStreamSynchronize(c->stream));   // nothing of an earlier call may still write the mirror
        hm->cycle = 0;
        k_solve_begin_lagged<<<1, 32, 0, c->stream>>>(c->d_scal, tol, maxcycles);
        KCHECK(c, "k_solve_begin_lagged");
        int launched = 0, known = 0;
        while (true) {
            while (launched < known + 2 && launched < maxcycles + 1) {
                if ((rc = run_cycle(c, p, b, true, true))) return rc;
                ++launched;
            }
            if ((rc = wait_cycle(c, known + 1))) return rc;
            hist[known] = ((volatile double*)c->h_hist)[known];
            nb = hm->nb;
            k = known++;
            if (!(hist[k] > tol * nb) || k >= maxcycles) break;
        }
        if (k == 0) {
            if ((rc = DISPATCH(c, remove_mean)(c, p))) return rc;
        } else {
            if ((rc = DISPATCH(c, apply_shift)(c, p))) return rc;
        }
    } else {
        if ((rc = DISPATCH(c, resnorm)(c, p, b))) return rc;
        k_solve_begin<<<1, 32, 0, c->stream>>>(c->d_scal, c->d_hist, tol, maxcycles);
        KCHECK(c, "k_solve_begin");
        if ((rc = read_scalars(c))) return rc;
        nb = c->h_scal->nb;
        hist[0] = bits_to_double(c->h_scal->absmax_bits[1]);
        const int depth = spec ? 2 : 1;
        hm->cycle = 0;
        int launched = 0;
        bool stop = !(maxcycles > 0 && hist[0] > tol * nb);
        while (!stop) {
            while (launched < maxcycles && launched - k < depth) {
                if ((rc = run_cycle(c, p, b, true, false))) return rc;
                ++launched;
            }
            if ((rc = wait_cycle(c, k + 1))) return rc;
            ++k;
            hist[k] = ((volatile double*)c->h_hist)[k];
            if (!(hist[k] > tol * nb) || k >= maxcycles) stop = true;
        }
        if (k == 0 && (rc = DISPATCH(c, remove_mean)(c, p))) return rc;
    }
    CU(c, cudaStreamSynchronize(c->stream));
    *ncycles = k;
    if (!isfinite(hist[k]) || !isfinite(nb)) return fail(c, WL_ENONFINITE, "wl_solve: the residual norm is not finite (NaN or Inf in p, b or the coefficients)");
    return (hist[k] > tol * nb) ? WL_NOT_CONVERGED : WL_OK;
}

// V-cycle-preconditioned conjugate gradients (oracle: ctx_solve_pcg).  One graph launch per iteration; the stop decision is
// taken on the device (last CTA of the x/r update) and mirrored to pinned host memory, which the host polls.
int solve_pcg_impl(wl_ctx* c, void* x, const void* b, double tol, int maxit, double* hist, int* nit, bool have_nb = false) {
    int rc;
    if ((rc = ensure_hist(c, maxit))) return rc;
    const size_t bytes = (size_t)c->lev[0].g.M * c->esz;
    for (int i = 0; i < 4; ++i)
        if (!c->cg_v[i]) {
            if (cudaMalloc(&c->cg_v[i], bytes) != cudaSuccess) { cudaGetLastError(); return fail(c, WL_ENOMEM, "wl_solve_pcg: cudaMalloc(work vector)"); }
            drop_graph(c);
        }
    if ((rc = DISPATCH(c, prepare)(c))) return rc;
    if (!have_nb && (rc = DISPATCH(c, absmax_b)(c, b))) return rc;
    volatile Scalars* hm = c->h_scal;
    CU(c, cudaStreamSynchronize(c->stream));   // nothing of an earlier call may still write the mirror
    hm->cycle = 0;
    hm->done = 0;
    k_pcg_begin<<<1, 32, 0, c->stream>>>(c->d_scal, tol, maxit);
    KCHECK(c, "k_pcg_begin");
    CU(c, cudaMemsetAsync(c->cg_v[2], 0, bytes, c->stream));   // p = 0: the first direction is z itself
    if ((rc = DISPATCH(c, pcg_residual)(c, x, b))) return rc;
    int k = 0;
    double nb = 0.0;
    while (true) {
        if ((rc = wait_cycle(c, k + 1))) return rc;
        if (hm->done == 2) break;                       // breakdown: the residual is exactly 0, no new entry
        hist[k] = ((volatile double*)c->h_hist)[k];
        nb = hm->nb;
        if (!(hist[k] > tol * nb) || k >= maxit) break;
        if ((rc = run_cycle(c, x, b, true, false, true))) return rc;
        ++k;
    }
    if (hm->done == 2) { --k; if (k < 0) k = 0; }
    if ((rc = DISPATCH(c, remove_mean)(c, x))) return rc;
    CU(c, cudaStreamSynchronize(c->stream));
    *nit = k;
    if (!isfinite(hist[k]) || !isfinite(nb)) return fail(c, WL_ENONFINITE, "wl_solve_pcg: the residual norm is not finite (NaN or Inf in p, b or the coefficients)");
    return (hist[k] > tol * nb) ? WL_NOT_CONVERGED : WL_OK;
}

// Fused (TMA) kernels need 16-byte aligned arrays; a misaligned caller array (e.g. a torch slice) sends its level to the
// generic kernels instead of failing in cuTensorMapEncodeTiled.
void note_alignment(wl_ctx* c, int level, std::initializer_list<const void*> ptrs) {
    uintptr_t bits = 0;
    for (const void* q : ptrs) bits |= (uintptr_t)q;
    c->unaligned = (bits & 15) != 0;
    c->unaligned_level = level;
}

int level_check(const wl_ctx* c, int level, bool need_next) {
    if (!c) return WL_EINVAL;
    if (level < 0 || level >= c->nlev) return WL_EINVAL;
    if (need_next && level + 1 >= c->nlev) return WL_EINVAL;
    return WL_OK;
}

}  // namespace

// ====================================================================================================================
extern "C" {

int wl_create(int ndim, const int64_t* dims, int dtype, wl_ctx** out) {
    if (out) *out = nullptr;
    if (!out || !dims) { snprintf(g_create_err, sizeof(g_create_err), "wl_create: null argument"); return WL_EINVAL; }
    if (dtype != WL_F32 && dtype != WL_F64) { snprintf(g_create_err, sizeof(g_create_err), "wl_create: bad dtype"); return WL_EINVAL; }
    if (ndim < 2 || ndim > 3) { snprintf(g_create_err, sizeof(g_create_err), "wl_create: ndim must be 2 or 3"); return WL_EDIMS; }
    long long cells = 1;
    for (int i = 0; i < ndim; ++i) {
        if (dims[i] < 4 || dims[i] > (1 << 20)) { snprintf(g_create_err, sizeof(g_create_err), "wl_create: every extent must be in [4, 2^20]"); return WL_EDIMS; }
        cells *= dims[i];
        if (cells > (1LL << 34)) { snprintf(g_create_err, sizeof(g_create_err), "wl_create: grid too large"); return WL_EDIMS; }
    }
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) { snprintf(g_create_err, sizeof(g_create_err), "wl_create: no CUDA device: %s", cudaGetErrorString(e)); return WL_ECUDA; }
    wl_ctx* c = new (std::nothrow) wl_ctx();
    if (!c) { snprintf(g_create_err, sizeof(g_create_err), "wl_create: out of host memory"); return WL_ENOMEM; }
    c->n = ndim;
    c->dtype = dtype;
    c->esz = (dtype == WL_F32) ? 4 : 8;
    cudaDeviceGetAttribute(&c->num_sms, cudaDevAttrMultiProcessorCount, dev);
    if (c->num_sms <= 0) c->num_sms = 148;

    long long N[3] = {dims[0], dims[1], ndim > 2 ? dims[2] : 1};
    int nlev = 0;
    while (true) {
        Level& v = c->lev[nlev];
        v.g.n = ndim;
        v.g.N0 = (int)N[0]; v.g.N1 = (int)N[1]; v.g.N2 = (int)N[2];
        v.g.M = N[0] * N[1] * N[2];
        ++nlev;
        bool ok = nlev < kMaxLevels;
        for (int i = 0; i < ndim; ++i)
            if (N[i] % 2 != 0 || N[i] / 2 < 4) ok = false;
        if (!ok) break;
        for (int i = 0; i < ndim; ++i) N[i] /= 2;
    }
    c->nlev = nlev;
    {   // coarse tail: the longest suffix of levels whose x ping-pong, b and L fit one CTA's shared memory
        size_t need = 0;
        c->tail_first = nlev;
        for (int l = nlev - 1; l >= 0 && nlev - l <= kTailMaxLevels; --l) {
            need += ((size_t)(4 + ndim) * c->lev[l].g.M * c->esz + 15) / 16 * 16;
            if (need > (size_t)kTailSmemBudget) break;
            c->tail_first = l;
        }
    }

    bool okm = true;
    auto dmalloc = [&](void** p, size_t bytes) {
        if (!okm) return;
        cudaError_t e2 = cudaMalloc(p, bytes < 16 ? 16 : bytes);
        if (e2 != cudaSuccess) { okm = false; snprintf(g_create_err, sizeof(g_create_err), "wl_create: cudaMalloc(%zu): %s", bytes, cudaGetErrorString(e2)); }
    };
    for (int l = 0; l < nlev; ++l) {
        Level& v = c->lev[l];
        dmalloc(&v.L, (size_t)v.g.M * ndim * c->esz);
        if (WL_FP64_C_PLANE && dtype == WL_F64 && ndim == 3) dmalloc(&v.C, (size_t)v.g.M * c->esz);   // read by the fp64 fused kernels only
        dmalloc(&v.x[1], (size_t)v.g.M * c->esz);
        if (l > 0) {
            dmalloc(&v.x[0], (size_t)v.g.M * c->esz);
            dmalloc(&v.b, (size_t)v.g.M * c->esz);
        }
    }
    dmalloc((void**)&c->d_scal, sizeof(Scalars));
    dmalloc((void**)&c->d_partials, sizeof(double) * kMaxPartials);
    if (okm && cudaMallocHost((void**)&c->h_scal, sizeof(Scalars)) != cudaSuccess) {
        okm = false;
        snprintf(g_create_err, sizeof(g_create_err), "wl_create: cudaMallocHost failed");
    }
    if (!okm) {
        cudaGetLastError();
        wl_destroy(c);
        return WL_ENOMEM;
    }
    cudaError_t e3 = cudaMemset(c->d_scal, 0, sizeof(Scalars));
    if (e3 == cudaSuccess) e3 = cudaStreamCreateWithFlags(&c->own_stream, cudaStreamNonBlocking);
    if (e3 == cudaSuccess) e3 = cudaEventCreateWithFlags(&c->ev_in, cudaEventDisableTiming);
    if (e3 == cudaSuccess) e3 = cudaEventCreateWithFlags(&c->ev_out, cudaEventDisableTiming);
    if (e3 != cudaSuccess) {   // not an allocation failure
        snprintf(g_create_err, sizeof(g_create_err), "wl_create: stream / event / memset: %s", cudaGetErrorString(e3));
        cudaGetLastError();
        wl_destroy(c);
        return WL_ECUDA;
    }
    if (DISPATCH(c, init_kernels)(c) != WL_OK) {
        snprintf(g_create_err, sizeof(g_create_err), "wl_create: %s", c->err);
        wl_destroy(c);
        return WL_ECUDA;
    }
    g_create_err[0] = 0;
    *out = c;
    return WL_OK;
}

void wl_destroy(wl_ctx* c) {
    if (!c) return;
    cudaStreamSynchronize(c->stream);
    drop_graph(c);
    if (c->own_stream) { cudaStreamSynchronize(c->own_stream); cudaStreamDestroy(c->own_stream); }
    if (c->copy_stream) { cudaStreamSynchronize(c->copy_stream); cudaStreamDestroy(c->copy_stream); }
    for (int i = 0; i < 3; ++i) if (c->ev_copy[i]) cudaEventDestroy(c->ev_copy[i]);
    if (c->ev_in) cudaEventDestroy(c->ev_in);
    if (c->ev_out) cudaEventDestroy(c->ev_out);
    for (int l = 0; l < kMaxLevels; ++l) {
        Level& v = c->lev[l];
        if (v.L) cudaFree(v.L);
        if (v.C) cudaFree(v.C);
        if (v.x[0]) cudaFree(v.x[0]);
        if (v.x[1]) cudaFree(v.x[1]);
        if (v.b) cudaFree(v.b);
        if (v.tmp) cudaFree(v.tmp);
        if (v.plan_items) cudaFree(v.plan_items);
        if (v.plan_start) cudaFree(v.plan_start);
    }
    if (c->d_scal) cudaFree(c->d_scal);
    if (c->d_partials) cudaFree(c->d_partials);
    if (c->d_hist) cudaFree(c->d_hist);
    if (c->h_hist) cudaFreeHost(c->h_hist);
    if (c->h_scal) cudaFreeHost(c->h_scal);
    if (c->b0) cudaFree(c->b0);
    if (c->d_bodies) cudaFree(c->d_bodies);
    if (c->h_bodies) cudaFreeHost(c->h_bodies);
    if (c->ev_bodies) cudaEventDestroy(c->ev_bodies);
    for (int i = 0; i < 4; ++i) if (c->cg_v[i]) cudaFree(c->cg_v[i]);
    if (c->stage_u) cudaFree(c->stage_u);
    if (c->stage_L) cudaFree(c->stage_L);
    if (c->stage_p) cudaFree(c->stage_p);
    cudaGetLastError();
    delete c;
}

int wl_set_stream(wl_ctx* c, void* s) {
    if (!c) return WL_EINVAL;
    if (c->stream != (cudaStream_t)s) drop_graph(c);
    c->pdl_armed = false;
    c->stream = (cudaStream_t)s;
    return WL_OK;
}

int wl_set_option(wl_ctx* c, int key, int value) {
    if (!c) return WL_EINVAL;
    drop_graph(c);
    switch (key) {
        case WL_OPT_FUSED: c->opt_fused = (value < 0 || value > 2) ? 1 : value; return WL_OK;
        case WL_OPT_GRAPH: c->opt_graph = value ? 1 : 0; return WL_OK;
        case WL_OPT_COARSE_CTA: c->opt_coarse_cta = value ? 1 : 0; return WL_OK;
        case WL_OPT_SOLVE_KERNELS: c->opt_solve_kernels = value ? 1 : 0; return WL_OK;
        case WL_OPT_SOLVER: c->opt_solver = value ? 1 : 0; return WL_OK;
        case WL_OPT_HOST_P_ZERO: c->opt_host_p_zero = value ? 1 : 0; return WL_OK;
        case WL_OPT_PDL: c->opt_pdl = value ? 1 : 0; return WL_OK;
        default: return fail(c, WL_EINVAL, "wl_set_option: unknown key");
    }
}

int wl_set_coeff(wl_ctx* c, const void* L) {
    if (!c) return WL_EINVAL;
    if (!L) return fail(c, WL_EINVAL, "wl_set_coeff: null L");
    return DISPATCH(c, set_coeff)(c, L);
}

int wl_set_bodies(wl_ctx* c, int nbodies, const double* bodies_host) {
    if (!c) return WL_EINVAL;
    if (nbodies < 0 || nbodies > kMaxBodies || (nbodies > 0 && !bodies_host)) return fail(c, WL_EINVAL, "wl_set_bodies: bad argument (at most 256 bodies)");
    for (int k = 0; k < nbodies; ++k) {
        const double* B = bodies_host + (size_t)k * kBodyDoubles;
        const int kind = (int)B[0];
        if ((kind != WL_BODY_SPHERE && kind != WL_BODY_TORUS) || (kind == WL_BODY_TORUS && c->n != 3) || !(B[4] >= 0.0) || !(B[5] >= 0.0))
            return fail(c, WL_EINVAL, "wl_set_bodies: bad body record");
    }
    if (!c->d_bodies && cudaMalloc((void**)&c->d_bodies, sizeof(double) * kMaxBodies * kBodyDoubles) != cudaSuccess) {
        cudaGetLastError();
        return fail(c, WL_ENOMEM, "wl_set_bodies: cudaMalloc");
    }
    if (!c->h_bodies) {
        if (cudaMallocHost((void**)&c->h_bodies, sizeof(double) * kMaxBodies * kBodyDoubles) != cudaSuccess) {
            cudaGetLastError();
            c->h_bodies = nullptr;
            return fail(c, WL_ENOMEM, "wl_set_bodies: cudaMallocHost");
        }
        CU(c, cudaEventCreateWithFlags(&c->ev_bodies, cudaEventDisableTiming));
    } else {
        CU(c, cudaEventSynchronize(c->ev_bodies));   // the previous call's upload has left the staging buffer
    }
    if (nbodies > 0) {
        // The records (at most 16 KB) go through a context-owned pinned buffer: with a pinned caller array the copy would be
        // truly asynchronous and a time stepper that moves its bodies for the next step would race with it.
        memcpy(c->h_bodies, bodies_host, sizeof(double) * (size_t)nbodies * kBodyDoubles);
        CU(c, cudaMemcpyAsync(c->d_bodies, c->h_bodies, sizeof(double) * (size_t)nbodies * kBodyDoubles, cudaMemcpyHostToDevice, c->stream));
    }
    CU(c, cudaEventRecord(c->ev_bodies, c->stream));
    return DISPATCH(c, set_bodies)(c, nbodies);
}

int wl_vcycle(wl_ctx* c, void* p, const void* b, double* rnorm_out) {
    if (!c) return WL_EINVAL;
    if (!p || !b) return fail(c, WL_EINVAL, "wl_vcycle: null pointer");
    if (!c->have_coeff) return fail(c, WL_ESTATE, "wl_vcycle: coefficients not set");
    note_alignment(c, 0, {p, b});
    int rc = run_cycle(c, p, b, false, false);
    if (rc) return rc;
    if (rnorm_out) {
        if ((rc = read_scalars(c))) return rc;
        *rnorm_out = bits_to_double(c->h_scal->absmax_bits[1]);
    }
    return WL_OK;
}

int wl_solve(wl_ctx* c, void* p, const void* b, double tol, int maxcycles, double* hist, int* ncycles) {
    if (!c) return WL_EINVAL;
    if (!p || !b || !hist || !ncycles || maxcycles < 0 || !(tol >= 0.0)) return fail(c, WL_EINVAL, "wl_solve: bad argument");
    if (!c->have_coeff) return fail(c, WL_ESTATE, "wl_solve: coefficients not set");
    note_alignment(c, 0, {p, b});
    return solve_impl(c, p, b, tol, maxcycles, hist, ncycles);
}

int wl_solve_pcg(wl_ctx* c, void* p, const void* b, double tol, int maxit, double* hist, int* nit) {
    if (!c) return WL_EINVAL;
    if (!p || !b || !hist || !nit || maxit < 0 || !(tol >= 0.0)) return fail(c, WL_EINVAL, "wl_solve_pcg: bad argument");
    if (!c->have_coeff) return fail(c, WL_ESTATE, "wl_solve_pcg: coefficients not set");
    note_alignment(c, 0, {p, b});
    return solve_pcg_impl(c, p, b, tol, maxit, hist, nit);
}

int wl_project(wl_ctx* c, void* u, const void* L, void* p, double tol, int maxcycles, double* hist, int* ncycles) {
    if (!c) return WL_EINVAL;
    if (!u || !p || !hist || !ncycles || maxcycles < 0 || !(tol >= 0.0)) return fail(c, WL_EINVAL, "wl_project: bad argument");
    int rc;
    if (L && (rc = DISPATCH(c, set_coeff)(c, L))) return rc;
    if (!c->have_coeff) return fail(c, WL_ESTATE, "wl_project: coefficients not set");
    if (!c->b0) {
        if (cudaMalloc(&c->b0, (size_t)c->lev[0].g.M * c->esz) != cudaSuccess) { cudaGetLastError(); return fail(c, WL_ENOMEM, "wl_project: cudaMalloc(b)"); }
    }
    note_alignment(c, 0, {p});
    if ((rc = DISPATCH(c, divergence)(c, u, c->b0, true))) return rc;
    int src = c->opt_solver ? solve_pcg_impl(c, p, c->b0, tol, maxcycles, hist, ncycles, true)
                            : solve_impl(c, p, c->b0, tol, maxcycles, hist, ncycles, true);
    if (src < 0) return src;
    if ((rc = DISPATCH(c, gradient)(c, u, p))) return rc;
    CU(c, cudaStreamSynchronize(c->stream));
    return src;
}

static int project_host_enqueue(wl_ctx* c, void* u_host, const void* L_host, void* p_host, double tol, int maxcycles, double* hist,
                                int* ncycles);

int wl_project_host(wl_ctx* c, void* u_host, const void* L_host, void* p_host, double tol, int maxcycles, double* hist,
                    int* ncycles) {
    if (!c) return WL_EINVAL;
    if (!u_host || !p_host || !hist || !ncycles || maxcycles < 0 || !(tol >= 0.0)) return fail(c, WL_EINVAL, "wl_project_host: bad argument");
    if (!L_host && !c->have_coeff) return fail(c, WL_ESTATE, "wl_project_host: coefficients not set");
    const int rc = project_host_enqueue(c, u_host, L_host, p_host, tol, maxcycles, hist, ncycles);
    if (rc < 0) {   // copies from / to the caller's buffers may be in flight on either stream: the caller may free them on return
        if (c->copy_stream) cudaStreamSynchronize(c->copy_stream);
        cudaStreamSynchronize(c->stream);
        cudaGetLastError();
    }
    return rc;
}

static int project_host_enqueue(wl_ctx* c, void* u_host, const void* L_host, void* p_host, double tol, int maxcycles, double* hist,
                                int* ncycles) {
    const size_t cell_bytes = (size_t)c->lev[0].g.M * c->esz;
    const size_t face_bytes = cell_bytes * c->n;
    if (!c->stage_u && cudaMalloc(&c->stage_u, face_bytes) != cudaSuccess) { cudaGetLastError(); return fail(c, WL_ENOMEM, "cudaMalloc(stage_u)"); }
    if (!c->stage_p && cudaMalloc(&c->stage_p, cell_bytes) != cudaSuccess) { cudaGetLastError(); return fail(c, WL_ENOMEM, "cudaMalloc(stage_p)"); }
    if (L_host && !c->stage_L && cudaMalloc(&c->stage_L, face_bytes) != cudaSuccess) { cudaGetLastError(); return fail(c, WL_ENOMEM, "cudaMalloc(stage_L)"); }
    if (!c->b0 && cudaMalloc(&c->b0, cell_bytes) != cudaSuccess) { cudaGetLastError(); return fail(c, WL_ENOMEM, "cudaMalloc(b)"); }
    if (!c->copy_stream) {
        if (cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking) != cudaSuccess ||
            cudaEventCreateWithFlags(&c->ev_copy[0], cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&c->ev_copy[1], cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&c->ev_copy[2], cudaEventDisableTiming) != cudaSuccess)
            return fail(c, WL_ECUDA, "wl_project_host: stream / event creation", cudaGetLastError());
    }
    cudaStream_t ms = c->stream, cs = c->copy_stream;
    int rc;
    // The copies that nothing waits for yet run on a second stream: L goes first and its hierarchy (H0) is built while u is
    // still crossing the bus; the pressure leaves while the gradient kernel runs.  One cudaMemcpyAsync per array.
    CU(c, cudaEventRecord(c->ev_copy[0], ms));                 // earlier work on the ctx stream may still use the staging buffers
    CU(c, cudaStreamWaitEvent(cs, c->ev_copy[0], 0));
    if (L_host) {
        CU(c, cudaMemcpyAsync(c->stage_L, L_host, face_bytes, cudaMemcpyHostToDevice, ms));
        if ((rc = DISPATCH(c, set_coeff)(c, c->stage_L))) return rc;
    }
    CU(c, cudaMemcpyAsync(c->stage_u, u_host, face_bytes, cudaMemcpyHostToDevice, cs));
    if (c->opt_host_p_zero) CU(c, cudaMemsetAsync(c->stage_p, 0, cell_bytes, cs));
    else CU(c, cudaMemcpyAsync(c->stage_p, p_host, cell_bytes, cudaMemcpyHostToDevice, cs));
    CU(c, cudaEventRecord(c->ev_copy[1], cs));
    CU(c, cudaStreamWaitEvent(ms, c->ev_copy[1], 0));
    note_alignment(c, 0, {c->stage_p});
    if ((rc = DISPATCH(c, divergence)(c, c->stage_u, c->b0, true))) return rc;
    int src = c->opt_solver ? solve_pcg_impl(c, c->stage_p, c->b0, tol, maxcycles, hist, ncycles, true)
                            : solve_impl(c, c->stage_p, c->b0, tol, maxcycles, hist, ncycles, true);
    if (src < 0) return src;
    CU(c, cudaEventRecord(c->ev_copy[2], ms));                 // p is final
    CU(c, cudaStreamWaitEvent(cs, c->ev_copy[2], 0));
    CU(c, cudaMemcpyAsync(p_host, c->stage_p, cell_bytes, cudaMemcpyDeviceToHost, cs));
    if ((rc = DISPATCH(c, gradient)(c, c->stage_u, c->stage_p))) return rc;
    CU(c, cudaMemcpyAsync(u_host, c->stage_u, face_bytes, cudaMemcpyDeviceToHost, ms));
    CU(c, cudaStreamSynchronize(ms));
    CU(c, cudaStreamSynchronize(cs));
    return src;
}

int wl_divergence(wl_ctx* c, const void* u, void* b) {
    if (!c) return WL_EINVAL;
    if (!u || !b) return fail(c, WL_EINVAL, "wl_divergence: null pointer");
    return DISPATCH(c, divergence)(c, u, b, false);
}

int wl_gradient(wl_ctx* c, void* u, const void* p) {
    if (!c) return WL_EINVAL;
    if (!u || !p) return fail(c, WL_EINVAL, "wl_gradient: null pointer");
    if (!c->have_coeff) return fail(c, WL_ESTATE, "wl_gradient: coefficients not set");
    return DISPATCH(c, gradient)(c, u, p);
}

int wl_convdiff(wl_ctx* c, const void* u, double nu, void* r) {
    if (!c) return WL_EINVAL;
    if (!u || !r || u == r) return fail(c, WL_EINVAL, "wl_convdiff: null or aliased pointer");
    return DISPATCH(c, convdiff)(c, u, nu, r);
}

int wl_jacobi(wl_ctx* c, int level, void* x, const void* b, int sweeps) {
    if (level_check(c, level, false)) return c ? fail(c, WL_EINVAL, "wl_jacobi: bad level") : WL_EINVAL;
    if (!x || !b || sweeps < 0) return fail(c, WL_EINVAL, "wl_jacobi: bad argument");
    if (!c->have_coeff) return fail(c, WL_ESTATE, "wl_jacobi: coefficients not set");
    return DISPATCH(c, jacobi)(c, level, x, b, c->lev[level].x[1], sweeps);
}

int wl_residual_restrict(wl_ctx* c, int level, const void* x, const void* b, void* bc) {
    if (level_check(c, level, true)) return c ? fail(c, WL_EINVAL, "wl_residual_restrict: bad level") : WL_EINVAL;
    if (!x || !b || !bc) return fail(c, WL_EINVAL, "wl_residual_restrict: null pointer");
    if (!c->have_coeff) return fail(c, WL_ESTATE, "wl_residual_restrict: coefficients not set");
    return DISPATCH(c, residual_restrict)(c, level, x, b, bc, nullptr);
}

int wl_prolong_correct(wl_ctx* c, int level, const void* xc, void* x) {
    if (level_check(c, level, true)) return c ? fail(c, WL_EINVAL, "wl_prolong_correct: bad level") : WL_EINVAL;
    if (!x || !xc) return fail(c, WL_EINVAL, "wl_prolong_correct: null pointer");
    return DISPATCH(c, prolong)(c, level, xc, x);
}

int wl_down(wl_ctx* c, int level, const void* x_in, const void* b, void* x_out, void* bc) {
    if (level_check(c, level, true)) return c ? fail(c, WL_EINVAL, "wl_down: bad level") : WL_EINVAL;
    if (!b || !x_out || x_in == x_out) return fail(c, WL_EINVAL, "wl_down: bad pointer");
    if (!c->have_coeff) return fail(c, WL_ESTATE, "wl_down: coefficients not set");
    if (c->opt_solve_kernels) { int rc = ensure_hist(c, 63); if (rc) return rc; }
    note_alignment(c, level, {x_in, b, x_out, bc});
    c->pdl_armed = false;
    c->solve_kernels_now = c->opt_solve_kernels;
    const int rc = DISPATCH(c, down)(c, level, x_in, b, x_out, bc ? bc : c->lev[level + 1].b);
    c->solve_kernels_now = 0;
    return rc;
}

int wl_up(wl_ctx* c, int level, const void* x_in, const void* xc, const void* b, void* x_out) {
    if (level_check(c, level, true)) return c ? fail(c, WL_EINVAL, "wl_up: bad level") : WL_EINVAL;
    if (!x_in || !b || !x_out || x_in == x_out) return fail(c, WL_EINVAL, "wl_up: bad pointer");
    if (!c->have_coeff) return fail(c, WL_ESTATE, "wl_up: coefficients not set");
    if (c->opt_solve_kernels) { int rc = ensure_hist(c, 63); if (rc) return rc; }
    note_alignment(c, level, {x_in, xc, b, x_out});
    c->pdl_armed = false;
    c->solve_kernels_now = c->opt_solve_kernels;
    const int rc = DISPATCH(c, up)(c, level, x_in, xc ? xc : c->lev[level + 1].x[1], b, x_out);
    c->solve_kernels_now = 0;
    return rc;
}

int wl_vcycle_level(wl_ctx* c, int level, void* x, const void* b) {
    if (level_check(c, level, false)) return c ? fail(c, WL_EINVAL, "wl_vcycle_level: bad level") : WL_EINVAL;
    if (!x || !b) return fail(c, WL_EINVAL, "wl_vcycle_level: null pointer");
    if (!c->have_coeff) return fail(c, WL_ESTATE, "wl_vcycle_level: coefficients not set");
    note_alignment(c, level, {x, b});
    c->pdl_armed = false;
    return DISPATCH(c, vcycle)(c, level, x, b, level == 0 ? c->lev[0].x[1] : c->lev[level].x[0], x);
}

int wl_residual_norm(wl_ctx* c, const void* p, const void* b, double* rnorm_out, double* mean_out) {
    if (!c) return WL_EINVAL;
    if (!p || !b || !rnorm_out) return fail(c, WL_EINVAL, "wl_residual_norm: null pointer");
    if (!c->have_coeff) return fail(c, WL_ESTATE, "wl_residual_norm: coefficients not set");
    int rc = DISPATCH(c, resnorm)(c, p, b);
    if (rc) return rc;
    if ((rc = read_scalars(c))) return rc;
    *rnorm_out = bits_to_double(c->h_scal->absmax_bits[1]);
    if (mean_out) *mean_out = c->h_scal->mean_p;
    return WL_OK;
}

int wl_selftest_recip(wl_ctx* c, uint64_t* mismatches_out, uint32_t* first_bad_bits_out) {
    if (!c) return WL_EINVAL;
    if (!mismatches_out) return fail(c, WL_EINVAL, "wl_selftest_recip: null pointer");
    // slots 2 and 3 of the context's scalars are scratch: [2] = mismatch count, [3] = smallest mismatching bit pattern
    const unsigned long long init[2] = {0ULL, ~0ULL};
    CU(c, cudaMemcpyAsync(&c->d_scal->absmax_bits[2], init, sizeof(init), cudaMemcpyHostToDevice, c->stream));
    k_selftest_recip<<<c->num_sms * 16, 256, 0, c->stream>>>(0x00800000u /* 2^-126 */, 0x7E800000u /* 2^126 */, &c->d_scal->absmax_bits[2]);
    KCHECK(c, "k_selftest_recip");
    unsigned long long res[2] = {0, 0};
    CU(c, cudaMemcpyAsync(res, &c->d_scal->absmax_bits[2], sizeof(res), cudaMemcpyDeviceToHost, c->stream));
    CU(c, cudaStreamSynchronize(c->stream));
    *mismatches_out = res[0];
    if (first_bad_bits_out) *first_bad_bits_out = res[0] ? (uint32_t)res[1] : 0u;
    return WL_OK;
}

int wl_selftest_fp32_rates(wl_ctx* c, double* out8) {
    if (!c) return WL_EINVAL;
    if (!out8) return fail(c, WL_EINVAL, "wl_selftest_fp32_rates: null pointer");
    // clocks of the timed loop per CTA land in the context's partials array (one CTA per SM, 16 warps each)
    constexpr int kWarps = 16, kIters = 4096;
    const int ctas = c->num_sms < kMaxPartials ? c->num_sms : kMaxPartials;
    long long* cyc = (long long*)c->d_partials;
    float* sink = (float*)&c->d_scal->absmax_bits[2];
    std::vector<long long> h((size_t)ctas);
    for (int mode = 0; mode < 4; ++mode) {
        for (int pass = 0; pass < 2; ++pass) {   // first pass warms the instruction cache
            const int it = pass ? kIters : 16;
            switch (mode) {
                case 0: k_fp32_rate<0><<<ctas, kWarps * 32, 0, c->stream>>>(sink, cyc, it, 1.0f); break;
                case 1: k_fp32_rate<1><<<ctas, kWarps * 32, 0, c->stream>>>(sink, cyc, it, 1.0f); break;
                case 2: k_fp32_rate<2><<<ctas, kWarps * 32, 0, c->stream>>>(sink, cyc, it, 1.0f); break;
                default: k_fp32_rate<3><<<ctas, kWarps * 32, 0, c->stream>>>(sink, cyc, it, 1.0f); break;
            }
            KCHECK(c, "k_fp32_rate");
        }
        CU(c, cudaMemcpyAsync(h.data(), cyc, sizeof(long long) * (size_t)ctas, cudaMemcpyDeviceToHost, c->stream));
        CU(c, cudaStreamSynchronize(c->stream));
        double avg = 0.0;
        for (int i = 0; i < ctas; ++i) avg += (double)h[(size_t)i];
        avg /= ctas;
        const bool packed = (mode & 1) != 0;
        const double winstr = (double)kWarps * kIters * (packed ? 8 : 16);
        out8[2 * mode] = winstr / avg;                               // warp-instructions per clock and SM
        out8[2 * mode + 1] = winstr * 32.0 * (packed ? 2 : 1) / avg;   // lane-operations (an fma counted once) per clock and SM
    }
    return WL_OK;
}

int wl_num_levels(const wl_ctx* c) { return c ? c->nlev : WL_EINVAL; }

int wl_level_dims(const wl_ctx* c, int level, int64_t* out) {
    if (!c || !out || level < 0 || level >= c->nlev) return WL_EINVAL;
    const Grid& g = c->lev[level].g;
    out[0] = g.N0;
    out[1] = g.N1;
    if (c->n > 2) out[2] = g.N2;
    return WL_OK;
}

int wl_get_coeff(const wl_ctx* c, int level, void* out) {
    if (!c || !out || level < 0 || level >= c->nlev) return WL_EINVAL;
    if (!c->have_coeff) return WL_ESTATE;
    const Level& v = c->lev[level];
    cudaError_t e = cudaMemcpyAsync(out, v.L, (size_t)v.g.M * c->n * c->esz, cudaMemcpyDeviceToDevice, c->stream);
    return e == cudaSuccess ? WL_OK : WL_ECUDA;
}

int64_t wl_launch_count(const wl_ctx* c) { return c ? c->launches : 0; }

int wl_plan_fused3d(const int64_t* dims, int dtype, int num_sms, int cap_items, int* items_out, int cap_ctas, int* start_out,
                    int* grid_out, int64_t* load_out) {
    if (!dims || (dtype != WL_F32 && dtype != WL_F64) || num_sms < 1) return WL_EINVAL;
    for (int i = 0; i < 3; ++i)
        if (dims[i] < 2 || dims[i] > (1 << 20)) return WL_EDIMS;
    if (dims[2] % 2) return WL_EDIMS;
    const Plan pl = (dtype == WL_F32) ? plan_fused3d((int)dims[0], (int)dims[1], (int)dims[2], Impl<float, 3>::FTX, Impl<float, 3>::FTY, num_sms)
                                      : plan_fused3d((int)dims[0], (int)dims[1], (int)dims[2], Impl<double, 3>::FTX, Impl<double, 3>::FTY, num_sms);
    if (grid_out) *grid_out = pl.grid();
    if (load_out) *load_out = pl.load;
    if (items_out && start_out && (int)pl.items.size() <= cap_items && pl.grid() + 1 <= cap_ctas) {
        for (size_t k = 0; k < pl.items.size(); ++k) {
            items_out[4 * k] = pl.items[k].X0; items_out[4 * k + 1] = pl.items[k].Y0;
            items_out[4 * k + 2] = pl.items[k].z0; items_out[4 * k + 3] = pl.items[k].nz;
        }
        for (size_t b = 0; b < pl.start.size(); ++b) start_out[b] = pl.start[b];
    }
    return (int)pl.items.size();
}

const char* wl_last_error(const wl_ctx* c) { return c ? c->err : g_create_err; }

}  // extern "C"
