// k_trace_tiled.cu -- tiled ray-trace writing phase to HBM (ao_trace_layers and the internal staging of the
// big-FFT sensors / science PSF): 32 x 256 output tiles, TMA-staged screen boxes, packed FFMA2 row march
// (trace_tile.cuh).  PAPER.md:56,60; reading O2.  Absolute phase: the FP64 piston sum is added back.
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <vector>

#include "trace_tile.cuh"
#include "trace2_plan.cuh"

namespace ao {

// ------------------------------------------------------------------------------------------------
// k_trace_tiled: the same tiled ray-trace, phase written to HBM (absolute: the FP64 piston sum is added back).
struct TiledTraceArgs {
    TraceArgs T;
    const int* sel; const long long* off; int n_sel;
    long long step_stride;
    int n_steps, tiles_x, tiles_y;
    float* phase;
};

__global__ void __launch_bounds__(kFusedThreads, 4)
k_trace_tiled(const TiledTraceArgs A)
{
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ TraceShared S;
    const int tid = threadIdx.x;
    const int k = (int)(blockIdx.x % (unsigned)A.n_steps);
    unsigned rest = blockIdx.x / (unsigned)A.n_steps;
    const int tx = (int)(rest % (unsigned)A.tiles_x); rest /= (unsigned)A.tiles_x;
    const int ty = (int)(rest % (unsigned)A.tiles_y);
    const int si = (int)(rest / (unsigned)A.tiles_y);
    const SourceP sp = A.T.srcs[A.sel[si]];
    const int jfirst = tx * kTileCols, ifirst = ty * kTraceRows;
    if (jfirst >= sp.N || ifirst >= sp.N) return;          // CTA-uniform
    u64 acc[kTraceRows];
    double refsum[2];
    trace_tile<kFusedThreads, 1>(A.T, sp, S, reinterpret_cast<float*>(smem), jfirst, ifirst, A.T.step0 + k, acc, refsum);
    float* out = A.phase + (size_t)k * A.step_stride + A.off[si];
    const int j0 = jfirst + tid, j1 = j0 + kFusedThreads;
#pragma unroll
    for (int i = 0; i < kTraceRows; ++i) {
        const int row = ifirst + i;
        if (row < sp.N) {
            const float2 f = unpack2(acc[i]);
            if (j0 < sp.N) out[(size_t)row * sp.N + j0] = (float)(((double)f.x + refsum[0]) * sp.scale);
            if (j1 < sp.N) out[(size_t)row * sp.N + j1] = (float)(((double)f.y + refsum[1]) * sp.scale);
        }
    }
}

// ------------------------------------------------------------------------------------------------
// k_trace_tiled2: two-step tiles of trace2.cuh (1/2 <= du <= 1: the NGS sensors and science directions, whose
// grids have the screen pitch, and the LGS sensors), phase written to HBM.  Absolute phase: the FP64 sum of the
// per-layer piston references is added back.
struct TiledTrace2Args {
    Trace2Args T;
    const int* sel; const long long* off; int n_sel;
    long long step_stride;
    int n_steps, n_pairs, tiles_x, tiles_y;
    float* phase;
};

template <int MODE>
__global__ void __launch_bounds__(kFusedThreads, 4)
k_trace_tiled2(const TiledTrace2Args A)
{
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ Trace2Shared S;
    const int tid = threadIdx.x;
    const int kp = (int)(blockIdx.x % (unsigned)A.n_pairs);
    unsigned rest = blockIdx.x / (unsigned)A.n_pairs;
    const int tx = (int)(rest % (unsigned)A.tiles_x); rest /= (unsigned)A.tiles_x;
    const int ty = (int)(rest % (unsigned)A.tiles_y);
    const int si = (int)(rest / (unsigned)A.tiles_y);
    const SourceP sp = A.T.srcs[A.sel[si]];
    const int jfirst = tx * kTileCols, ifirst = ty * kTR;
    if (jfirst >= sp.N || ifirst >= sp.N) return;          // CTA-uniform
    u64 acc[kKS * kTR];
    double refsum[2];
    trace2_tile<kFusedThreads, true, MODE>(A.T, sp, S, smem, jfirst, ifirst, A.T.step0 + 2 * kp, acc, refsum);
    const int j0 = jfirst + tid, j1 = j0 + kFusedThreads;
#pragma unroll
    for (int s = 0; s < kKS; ++s) {
        const int k = 2 * kp + s;
        if (k >= A.n_steps) break;
        float* out = A.phase + (size_t)k * A.step_stride + A.off[si];
#pragma unroll
        for (int i = 0; i < kTR; ++i) {
            const int row = ifirst + i;
            if (row < sp.N) {
                const float2 f = unpack2(acc[s * kTR + i]);
                if (j0 < sp.N) out[(size_t)row * sp.N + j0] = (float)(((double)f.x + refsum[0]) * sp.scale);
                if (j1 < sp.N) out[(size_t)row * sp.N + j1] = (float)(((double)f.y + refsum[1]) * sp.scale);
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------
// host side
struct TilePlan { bool ok; int pitch, rows, ns; size_t smem; };

// Staging plan of the tiled ray-trace for the sources `src` (all active layers): the box of a 32 x 256 tile
// must fit the shared-memory stages and the row march needs 0 < du <= 1.  `min_bytes`: floor on the dynamic
// shared memory (the exchange buffer of k_fused).
static TilePlan plan_tiles(const ao_geometry* g, const std::vector<int>& src, size_t min_bytes)
{
    TilePlan pl = {false, 0, 0, 0, 0};
    double du_max = 0.0;
    int s_min = 1 << 30;
    for (int s : src) {
        const SourceP& sp = g->sources[s];
        for (const LayerP& lp : g->layers) {
            if (!(lp.height < sp.H)) continue;
            double du = (1.0 - lp.height * sp.inv_H) * sp.d * lp.inv_pitch;
            if (fabs(du - 1.0) < 1e-9) du = 1.0;
            if (!(du > 0.0) || du > 1.0) return pl;              // the row march assumes 0 < du <= 1
            if (lp.S % 4 != 0) return pl;                          // 16-byte aligned rows for the bulk copies
            if (du > du_max) du_max = du;
            if (lp.S < s_min) s_min = lp.S;
        }
    }
    if (du_max == 0.0) { du_max = 1.0; s_min = 1 << 30; }          // no active layer at all: any plan works
    pl.pitch = (((int)ceil((kTileCols - 1) * du_max) + 7) + 3) & ~3;
    pl.rows = (int)ceil((kTraceRows - 1) * du_max) + 3 + 1;       // box rows + one prefetch pad row
    if (s_min < pl.pitch || s_min < pl.rows) return pl;            // a box row may wrap the screen edge once only
    const size_t stage = (size_t)pl.rows * pl.pitch * sizeof(float);
    // 4 CTAs per SM need <= ~48 KB of dynamic shared memory each; prefer 3 stages when they fit
    pl.ns = (3 * stage <= 48 * 1024) ? 3 : 2;
    if (const char* ev = getenv("AO_FUSED_STAGES")) { const int v = atoi(ev); if (v >= 2 && v <= kTraceMaxStages) pl.ns = v; }
    pl.smem = pl.ns * stage;
    if (pl.smem < min_bytes) pl.smem = min_bytes;
    pl.smem += 128;
    pl.ok = pl.smem <= 200 * 1024;
    return pl;
}

static TraceArgs make_trace_args(const ao_geometry* g, const TilePlan& pl, int64_t step0, double dt)
{
    TraceArgs t;
    t.layers = g->d_layers; t.n_layers = (int)g->layers.size(); t.srcs = g->d_sources;
    t.step0 = (long long)step0; t.dt = dt; t.pitch = pl.pitch; t.rows = pl.rows; t.ns = pl.ns;
    return t;
}

// Tiled ray-trace of a source group into a phase buffer; cudaErrorNotSupported if the geometry is outside
// the fast path (the caller then uses the per-sample kernel of k_trace.cu).
cudaError_t launch_trace_tiled(ao_geometry* g, const Group& grp, bool api_layout, long long step_stride,
                               int64_t step0, int n_steps, double dt, float* phase, cudaStream_t st)
{
    const int n_sel = (int)grp.src.size();
    if (n_sel == 0 || n_steps <= 0) return cudaSuccess;
    const Tile2Plan p2 = plan_tiles2(g, grp.src, dt, 0);
    if (p2.ok && !getenv("AO_TRACE_OLD")) {
        auto kern2 = !p2.anydu ? k_trace_tiled2<0> : (p2.quad ? k_trace_tiled2<2> : k_trace_tiled2<1>);
        cudaError_t e2 = cudaFuncSetAttribute(kern2, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p2.smem);
        if (e2 != cudaSuccess) return e2;
        TiledTrace2Args a;
        a.T = make_trace2_args(g, p2, step0, dt);
        a.sel = grp.d_src; a.off = api_layout ? grp.d_off_api : grp.d_off_stage; a.n_sel = n_sel;
        a.step_stride = step_stride;
        a.tiles_x = (grp.max_N + kTileCols - 1) / kTileCols;
        a.tiles_y = (grp.max_N + kTR - 1) / kTR;
        const long long per_pair = (long long)a.tiles_x * a.tiles_y * n_sel;
        int max_steps = (int)std::max<long long>(2, 2 * (0x7fffffffLL / per_pair));
        max_steps &= ~1;
        for (int k0 = 0; k0 < n_steps; k0 += max_steps) {
            const int ks = n_steps - k0 < max_steps ? n_steps - k0 : max_steps;
            TiledTrace2Args b = a;
            b.T.step0 = (long long)step0 + k0; b.n_steps = ks; b.n_pairs = (ks + kKS - 1) / kKS;
            b.phase = phase + (size_t)k0 * step_stride;
            kern2<<<(unsigned)(per_pair * b.n_pairs), kFusedThreads, p2.smem, st>>>(b);
            g->launches++;
            if ((e2 = cudaGetLastError()) != cudaSuccess) return e2;
        }
        return cudaSuccess;
    }
    const TilePlan pl = plan_tiles(g, grp.src, 0);
    if (!pl.ok) return cudaErrorNotSupported;
    cudaError_t e = cudaFuncSetAttribute(k_trace_tiled, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl.smem);
    if (e != cudaSuccess) return e;
    TiledTraceArgs a;
    a.T = make_trace_args(g, pl, step0, dt);
    a.sel = grp.d_src; a.off = api_layout ? grp.d_off_api : grp.d_off_stage; a.n_sel = n_sel;
    a.step_stride = step_stride;
    a.tiles_x = (grp.max_N + kTileCols - 1) / kTileCols;
    a.tiles_y = (grp.max_N + kTraceRows - 1) / kTraceRows;
    const long long per_step = (long long)a.tiles_x * a.tiles_y * n_sel;
    const int max_steps = (int)std::max<long long>(1, 0x7fffffffLL / per_step);
    for (int k0 = 0; k0 < n_steps; k0 += max_steps) {
        const int ks = n_steps - k0 < max_steps ? n_steps - k0 : max_steps;
        TiledTraceArgs b = a;
        b.T.step0 = (long long)step0 + k0; b.n_steps = ks;
        b.phase = phase + (size_t)k0 * step_stride;
        k_trace_tiled<<<(unsigned)(per_step * ks), kFusedThreads, pl.smem, st>>>(b);
        g->launches++;
        if ((e = cudaGetLastError()) != cudaSuccess) return e;
    }
    return cudaSuccess;
}

}  // namespace ao
