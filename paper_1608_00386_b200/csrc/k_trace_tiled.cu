// k_trace_tiled.cu -- tiled ray-trace writing phase to HBM (ao_trace_layers and the internal staging of the
// big-FFT sensors / science PSF): two-step tiles of 16 x 256 samples, TMA-staged screen boxes, packed FFMA2 row
// marches (trace2.cuh).  PAPER.md:56,60; reading O2.  Absolute phase: the FP64 piston sum is added back.
// Geometries outside the plan (boxes too large for shared memory, screen sides not a multiple of 4) return
// cudaErrorNotSupported and the caller uses the per-sample kernel of k_trace.cu.
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <vector>

#include "trace2_plan.cuh"

namespace ao {

// ------------------------------------------------------------------------------------------------
// k_trace_tiled2: two-step tiles of trace2.cuh, phase written to HBM.  MODE selects the row march: 0 three-term
// (every layer has 1/2 <= du <= 1: the NGS sensors and science directions, whose grids have the screen pitch, and the
// c2-c4 LGS sensors at M = 32), 2 quad (every layer du <= 2/3: the fine LGS grid of M = 64), 1 two-row (anything else).
// Absolute phase: the FP64 sum of the per-layer piston references is added back.
struct TiledTrace2Args {
    Trace2Args T;
    const int* sel; const long long* off; int n_sel;
    long long step_stride;
    int n_steps, n_pairs, tiles_x, tiles_y;
    float* phase;
};

template <int MODE>
__global__ void __launch_bounds__(kFusedThreads, 3)
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
    const bool in0 = j0 < sp.N, in1 = j1 < sp.N;
    const int rows_in = min(kTR, sp.N - ifirst);          // CTA-uniform
    const double scale = sp.scale;
#pragma unroll
    for (int s = 0; s < kKS; ++s) {
        const int k = 2 * kp + s;
        if (k >= A.n_steps) break;
        float* out = A.phase + (size_t)k * A.step_stride + A.off[si] + (size_t)ifirst * sp.N;
        if (sp.map == nullptr) {
#pragma unroll
            for (int i = 0; i < kTR; ++i) {
                if (i < rows_in) {
                    const float2 f = unpack2(acc[s * kTR + i]);
                    if (in0) out[(size_t)i * sp.N + j0] = (float)(((double)f.x + refsum[0]) * scale);
                    if (in1) out[(size_t)i * sp.N + j1] = (float)(((double)f.y + refsum[1]) * scale);
                }
            }
        } else {
            const float* mp = sp.map + (size_t)ifirst * sp.N;
#pragma unroll
            for (int i = 0; i < kTR; ++i) {
                if (i < rows_in) {
                    const float2 f = unpack2(acc[s * kTR + i]);
                    if (in0) out[(size_t)i * sp.N + j0] = (float)(((double)f.x + refsum[0]) * scale + (double)__ldg(mp + (size_t)i * sp.N + j0));
                    if (in1) out[(size_t)i * sp.N + j1] = (float)(((double)f.y + refsum[1]) * scale + (double)__ldg(mp + (size_t)i * sp.N + j1));
                }
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------
// host side
// Tiled ray-trace of a source group into a phase buffer; cudaErrorNotSupported if the geometry is outside
// the fast path (the caller then uses the per-sample kernel of k_trace.cu).
cudaError_t launch_trace_tiled(ao_geometry* g, const Group& grp, bool api_layout, long long step_stride,
                               int64_t step0, int n_steps, double dt, float* phase, cudaStream_t st)
{
    const int n_sel = (int)grp.src.size();
    if (n_sel == 0 || n_steps <= 0) return cudaSuccess;
    // the phase writer has no exchange buffer to alias: three CTAs per SM (75 KB each) buy a third stage for the wide
    // boxes of same-pitch grids (NGS sensors, science directions: du = 1, 22 KB per stage)
    const Tile2Plan p2 = plan_tiles2(g, grp.src, dt, 0, 75 * 1024);
    if (p2.ok) {
        auto kern2 = p2.unit ? k_trace_tiled2<3> : !p2.anydu ? k_trace_tiled2<0> : (p2.quad ? k_trace_tiled2<2> : k_trace_tiled2<1>);
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
    return cudaErrorNotSupported;
}

}  // namespace ao
