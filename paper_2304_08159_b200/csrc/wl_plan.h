// wl_plan.h — host-side work split of one fused 3-D level half (DESIGN.md §6.1 "Work split").  Plain C++, no CUDA.
//
// A launch is one persistent CTA per SM; a work item is (tile, z-range) and costs nz + RI plane steps, RI = 9: 6 run-in steps
// of the three skewed stencil stages + about 3 steps' worth of pipeline fill (TMA latency at the item's start, the join at its
// end; RI = 6, 9, 12 measured on the 256^3 and 512^3 levels: 9 is the fastest).  The plan gives every CTA an explicit list of
// items so that
//   * the largest per-CTA load  sum(nz + RI)  is as small as possible (the launch ends with its slowest CTA), and
//   * CTAs that run at the same time work on neighbouring tiles of the same z-range in lockstep (a halo fetched by one is
//     still in L2 when its neighbour asks).
// Two families are searched and the cheaper one is taken:
//   uniform  z cut into nc equal chunks, the nc * ntiles items dealt round-robin, chunk-major (round 1's split);
//   groups   z cut into UNEQUAL chunks, chunk c owned by its own group of g_c CTAs that deal its ntiles items round-robin, m_c =
//            ceil(ntiles / g_c) items per CTA: a chunk of a group with more items per CTA is shorter, so that all groups end
//            together.  For a load T a group of multiplicity m uses ceil(ntiles / m) CTAs and covers floor((T / m - RI) / 2)
//            plane pairs: an unbounded knapsack over the CTA count gives the largest z-extent reachable with T, a bisection
//            on T the smallest feasible load.  256^3 on 148 SMs: 64 tiles; uniform = 2 chunks x 64 tiles = 128 CTAs x (128 + RI)
//            steps (20 SMs idle); groups = 118 + 116 planes on 64 CTAs each and 22 planes on 16 CTAs x 4 tiles: 118 + RI.
#pragma once
#include <algorithm>
#include <vector>

namespace wl {

struct PlanItem { int X0, Y0, z0, nz; };   // tile origin (cells), first plane (even), planes (even, >= 2)

struct Plan {
    std::vector<PlanItem> items;   // grouped by CTA
    std::vector<int> start;        // CTA b owns items [start[b], start[b + 1]); size = grid + 1
    long long load = 0;            // largest per-CTA sum of (nz + WL_PLAN_RUNIN)
    int grid() const { return (int)start.size() - 1; }
};

#ifndef WL_PLAN_RUNIN
#define WL_PLAN_RUNIN 9
#endif
inline Plan plan_fused3d(int N0, int N1, int N2, int TX, int TY, int num_sms) {
    constexpr int RI = WL_PLAN_RUNIN;
    const int tiles_x = (N0 + TX - 1) / TX, tiles_y = (N1 + TY - 1) / TY;
    const int n = tiles_x * tiles_y;
    const int H = N2 / 2;                       // plane pairs
    const int G = num_sms < 1 ? 1 : num_sms;
    auto tile_item = [&](int tile, int z0, int nz) {
        const int tyi = tile / tiles_x, txi = tile - tyi * tiles_x;
        return PlanItem{txi * TX, tyi * TY, z0, nz};
    };
    auto finish = [&](std::vector<std::vector<PlanItem>>& per) {
        Plan p;
        p.start.push_back(0);
        for (auto& v : per) {
            long long ld = 0;
            for (auto& it : v) { p.items.push_back(it); ld += it.nz + RI; }
            p.load = std::max(p.load, ld);
            p.start.push_back((int)p.items.size());
        }
        return p;
    };

    // ---- uniform chunks ---------------------------------------------------------------------------------------------
    Plan best;
    {
        long long best_cost = -1;
        int best_nc = 1;
        for (int nc = 1; nc <= H && nc <= 4096; ++nc) {
            const long long items = (long long)n * nc;
            const long long waves = (items + G - 1) / G;
            const long long cost = waves * (2LL * ((H + nc - 1) / nc) + RI);
            if (best_cost < 0 || cost < best_cost) { best_cost = cost; best_nc = nc; }
        }
        const long long items = (long long)n * best_nc;
        const int grid = (int)std::min<long long>(items, G);
        std::vector<std::vector<PlanItem>> per(grid);
        for (long long it = 0; it < items; ++it) {
            const int chunk = (int)(it / n), tile = (int)(it - (long long)chunk * n);
            const int z0 = (int)(((long long)H * chunk / best_nc) << 1);
            const int z1 = (int)(((long long)H * (chunk + 1) / best_nc) << 1);
            per[it % grid].push_back(tile_item(tile, z0, z1 - z0));
        }
        best = finish(per);
    }

    // ---- groups with unequal chunks -------------------------------------------------------------------------------------
    {
        const int mmax = std::min(n, 64);
        std::vector<int> choice;                       // multiplicities of the chosen groups
        auto cover = [&](long long T, std::vector<int>* out) -> long long {
            // best[k] = most plane pairs coverable with k CTAs; from[k] = multiplicity of the last group (0: none)
            std::vector<long long> bestk(G + 1, 0);
            std::vector<int> from(G + 1, 0);
            for (int k = 1; k <= G; ++k) {
                bestk[k] = bestk[k - 1];
                from[k] = -1;                          // -1: CTA k unused
                for (int m = 1; m <= mmax; ++m) {
                    const int g = (n + m - 1) / m;
                    const long long h = (T / m - RI) / 2;
                    if (g > k || h < 1) continue;
                    if (bestk[k - g] + h > bestk[k]) { bestk[k] = bestk[k - g] + h; from[k] = m; }
                }
            }
            if (out) {
                out->clear();
                for (int k = G; k > 0;) {
                    if (from[k] <= 0) { --k; continue; }
                    out->push_back(from[k]);
                    k -= (n + from[k] - 1) / from[k];
                }
            }
            return bestk[G];
        };
        long long lo = 8, hi = best.load;              // smallest T whose cover reaches H
        if (cover(hi, nullptr) >= H) {
            while (lo < hi) {
                const long long mid = (lo + hi) / 2;
                if (cover(mid, nullptr) >= H) hi = mid; else lo = mid + 1;
            }
            cover(hi, &choice);
            std::vector<long long> h(choice.size());
            long long tot = 0;
            for (size_t c = 0; c < choice.size(); ++c) { h[c] = (hi / choice[c] - RI) / 2; tot += h[c]; }
            while (tot > H) {                          // trim the excess off the heaviest group that can spare a pair
                size_t w = choice.size();
                for (size_t c = 0; c < choice.size(); ++c)
                    if (h[c] > 1 && (w == choice.size() || choice[c] * (2 * h[c] + RI) > choice[w] * (2 * h[w] + RI))) w = c;
                if (w == choice.size()) break;
                --h[w]; --tot;
            }
            if (tot == H) {
                std::vector<std::vector<PlanItem>> per;
                int z0 = 0;
                for (size_t c = 0; c < choice.size(); ++c) {
                    const int m = choice[c], g = (n + m - 1) / m, nz = (int)(2 * h[c]);
                    const size_t base = per.size();
                    per.resize(base + g);
                    for (int tile = 0; tile < n; ++tile) per[base + tile % g].push_back(tile_item(tile, z0, nz));
                    z0 += nz;
                }
                Plan p = finish(per);
                if (p.load < best.load) best = p;
            }
        }
    }
    return best;
}

}  // namespace wl
