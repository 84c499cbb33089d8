// trace2_plan.cuh -- host-side staging plan of the two-step tiled ray-trace (trace2.cuh), shared by the fused
// WFS kernel (k_fused.cu) and the tiled phase writer (k_trace_tiled.cu).
#pragma once
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <vector>

#include "trace2.cuh"

namespace ao {

constexpr int kFusedThreads = 128;
constexpr int kTileCols = 2 * kFusedThreads;

struct Tile2Plan { bool ok; int pitch, rows, ns; size_t smem; int anydu, quad, unit, tma; };

// Staging plan of the two-step tiled ray-trace for the sources `src` (all active layers): the union box of a
// 16 x 256 tile over two consecutive steps must fit a shared-memory stage.  Layers with 1/2 <= du <= 1 (screen
// pixels per output sample) take the three-term row march; if any layer is outside, the two-row march runs.  `min_bytes`: floor on the stage region (the exchange buffer of k_fused aliases it).
inline Tile2Plan plan_tiles2(const ao_geometry* g, const std::vector<int>& src, double dt, size_t min_bytes,
                             size_t budget = 55 * 1024 + 512, bool want_tma = false)
{
    Tile2Plan pl = {false, 0, 0, 0, 0, 0, 0, 0, 0};
    double du_max = 0.0;
    bool all_unit = true;
    double ext_x = 0.0, ext_y = 0.0;                               // box extent beyond the taps, screen pixels
    int s_min = 1 << 30;
    bool any = false;
    for (int s : src) {
        const SourceP& sp = g->sources[s];
        for (const LayerP& lp : g->layers) {
            if (!(lp.height < sp.H)) continue;
            double du = (1.0 - lp.height * sp.inv_H) * sp.d * lp.inv_pitch;
            if (fabs(du - 1.0) < 1e-9) du = 1.0;
            if (!(du > 0.0) || du > 8.0) return pl;               // absurd sampling ratio: not this path
            if (du < 0.5 || du > 1.0) pl.anydu = 1;                // outside the three-term march: two-row march
            if (du > du_max) du_max = du;
            if (du != 1.0) all_unit = false;
            if (lp.S % 4 != 0 || ((uintptr_t)lp.screen & 15) != 0) return pl;   // 16-byte aligned rows for the bulk copies
            const double shx = fabs(lp.wx * dt * lp.inv_pitch) * (kKS - 1), shy = fabs(lp.wy * dt * lp.inv_pitch) * (kKS - 1);
            ext_x = std::max(ext_x, (kTileCols - 1) * du + shx);
            ext_y = std::max(ext_y, (kTR - 1) * du + shy);
            if (lp.S < s_min) s_min = lp.S;
            any = true;
        }
    }
    if (!any) { ext_x = kTileCols - 1; ext_y = kTR - 1; }
    if (!(ext_x < 4096.0 && ext_y < 4096.0)) return pl;            // absurd wind shift per step: not this path
    pl.pitch = (((int)ceil(ext_x) + 8) + 3) & ~3;                  // + alignment (3), right tap, rounding slack
    pl.quad = (pl.anydu && du_max <= 0.66) ? 1 : 0;                // every layer has du <= 2/3: groups of four rows
    if (any && all_unit && pl.pitch <= kUnitPitch) { pl.unit = 1; pl.pitch = kUnitPitch; }   // du = 1: table-free march
    pl.rows = (int)ceil(ext_y) + 3 + 1 + (pl.quad ? 2 : 0);        // box rows + one pad row (+ the quad march's fourth row)
    if (want_tma && any && !pl.unit) {
        // tensor-map copies: box {pitch, rows} <= 256 x 256, stages 128-byte aligned (rows * pitch a multiple of 32 floats)
        const int pt = (pl.pitch + 7) & ~7, rw = (pl.rows + 3) & ~3;
        if (pt <= 256 && rw <= 256) { pl.tma = 1; pl.pitch = pt; pl.rows = rw; }
    }
    if (s_min < pl.pitch || s_min < pl.rows) return pl;            // a box row may wrap the screen edge once only
    const size_t stage = (size_t)pl.rows * pl.pitch * sizeof(float);
    const size_t sched = trace2_sched_bytes((int)g->layers.size());
    // fused kernel: 4 CTAs per SM, <= ~55 KB of shared memory each; as many stages (<= 4) as fit the budget, at least 2
    pl.ns = 2;
    while (pl.ns < kT2MaxStages && (pl.ns + 1) * stage + sched + 128 + 256 <= budget) ++pl.ns;
#ifdef AO_PROFILE_SWITCHES      // profiling builds only: override the stage count
    if (const char* ev = getenv("AO_FUSED_STAGES")) { const int v = atoi(ev); if (v >= 2 && v <= kT2MaxStages) pl.ns = v; }
#endif
    size_t region = pl.ns * stage;
    if (region < min_bytes) region = (min_bytes + 15) & ~(size_t)15;
    pl.smem = region + sched + 128;
    pl.ok = pl.smem <= 200 * 1024;
    return pl;
}

inline Trace2Args make_trace2_args(const ao_geometry* g, const Tile2Plan& pl, int64_t step0, double dt)
{
    Trace2Args t;
    t.layers = g->d_layers; t.n_layers = (int)g->layers.size(); t.srcs = g->d_sources;
    t.step0 = (long long)step0; t.dt = dt; t.pitch = pl.pitch; t.rows = pl.rows; t.ns = pl.ns;
    t.tmaps = nullptr;
#ifdef AO_PROFILE_SWITCHES      // profiling builds only (AO_BUILD_PROFILE=1): switch parts of the kernel off, results are wrong
    { const char* ev = getenv("AO_DBG"); t.dbg = ev ? atoi(ev) : 0; }
#endif
    return t;
}

}  // namespace ao
