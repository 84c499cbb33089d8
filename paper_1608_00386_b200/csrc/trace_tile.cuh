// trace_tile.cuh -- the tiled ray-trace device routine shared by k_fused (trace + SH + CoG) and
// k_trace_tiled (trace -> phase buffer).  PAPER.md:56 (frozen flow), PAPER.md:60 (open-loop wavefront of
// every star, finite-distance projection of the LGS); reading O2 of DESIGN.md section 3.
//
// A CTA of NT threads produces a tile of 32 output rows x 2 NT output columns of one (step, source).
// Per layer the screen footprint of the tile (a box of <= 31 du + 3 rows by <= (2 NT - 1) du + 7 columns,
// 0 < du <= 1 the screen pixels per output sample) is staged in shared memory by the TMA engine: the lanes
// of warp 0 issue one cp.async.bulk row copy each (two when the row crosses the periodic edge of the
// screen), completing on a "full" mbarrier; `ns` stages are in flight; a stage is handed back through an
// "empty" mbarrier on which every warp arrives when it has consumed the layer, so the layer loop has no
// CTA-wide barrier.
//
// Each thread owns two columns (tid and tid + NT) packed in one 64-bit register pair, so that every
// floating-point instruction of the inner loop is a packed FFMA2 / FADD2 (sm_100 f32x2).  Bilinear
// interpolation is separable: the x-interpolated screen rows X_r = s[r][j0] + fx (s[r][j0+1] - s[r][j0])
// are computed once per screen row, and an output row costs two FFMA2: acc_i += (1-fy_i) X_r + fy_i X_{r+1}.
// Because du <= 1 an output row needs at most one new screen row: the per-row decision "advance" and the
// weights (1-fy_i, fy_i) are warp-uniform and are precomputed per (CTA, layer) by warp 0 in FP64 into a
// shared-memory schedule (one LDS.128 per row); the taps of the next screen row are prefetched one advance
// ahead.  Precision: column coordinates are FP64 per (thread, layer), so cell and fraction are exact at
// screen coordinates of several thousand pixels; a per-thread-group piston reference (the first tap of the
// group's first column) is subtracted from every tap so that the fp32 sums stay at the few-radian level;
// its FP64 sum is returned so that callers that need absolute phase can add it back.
#pragma once
#include "ao_device.cuh"
#include "pk_tma.cuh"

namespace ao {

constexpr int kTraceRows = 32;          // output rows of a tile
constexpr int kTraceMaxStages = 4;

struct TraceArgs {
    const LayerP* layers; int n_layers;
    const SourceP* srcs;
    long long step0; double dt;
    int pitch;            // staged row pitch in floats (multiple of 4)
    int rows;             // staged rows allocated per stage (box rows + 1 prefetch pad row)
    int ns;               // stages in flight (2 or 3)
};

struct __align__(16) TraceShared {
    float4 sched[kTraceMaxStages][kTraceRows];      // per row: (1-fy, fy, advance flag, unused)
    uint64_t full_bar[kTraceMaxStages], empty_bar[kTraceMaxStages];
    double u0[kMaxLayers], du[kMaxLayers], v0[kMaxLayers], c0[kMaxLayers];
    int wt[kMaxLayers], rt[kMaxLayers], act[kMaxLayers];
    int nact;
};

// The 32 output rows of a layer as a two-state machine.  The x-interpolated screen rows above and below
// the current output row live in the packed registers Xa and Xb; in state E the top row is Xa and the
// bottom row Xb, in state O the roles are swapped, so that advancing one screen row (new bottom row ->
// the register of the old top row) needs no register move: it just changes state.  The advance decision
// comes from the shared-memory schedule and is warp-uniform.  The taps of the next screen row are
// prefetched one advance ahead (p0 = left taps, p1 = right taps of the two columns).
#define AO_TRACE_ADV(XNEW)                                                                       \
    XNEW = fma2(fx, sub2(p1, p0), sub2(p0, ref));                                                \
    tp0 += pb; tp1 += pb;                                                                        \
    p0 = pack2(lds_f32(tp0), lds_f32(tp1));                                                      \
    p1 = pack2(lds_f32_next(tp0), lds_f32_next(tp1));
#define AO_TRACE_ACC(i, XTOP, XBOT)                                                              \
    acc[i] = fma2(pack2(sc.y, sc.y), XBOT, fma2(pack2(sc.x, sc.x), XTOP, acc[i]));
#define AO_TRACE_ROW(i, inext)                                                                   \
    LE_##i: {                                                                                    \
        const float4 sc = sch[i];                                                                \
        if (__float_as_int(sc.z) != 0) { AO_TRACE_ADV(Xa) AO_TRACE_ACC(i, Xb, Xa) goto LO_##inext; } \
        AO_TRACE_ACC(i, Xa, Xb) goto LE_##inext;                                                 \
    }                                                                                            \
    LO_##i: {                                                                                    \
        const float4 sc = sch[i];                                                                \
        if (__float_as_int(sc.z) != 0) { AO_TRACE_ADV(Xb) AO_TRACE_ACC(i, Xa, Xb) goto LE_##inext; } \
        AO_TRACE_ACC(i, Xb, Xa) goto LO_##inext;                                                 \
    }
#define AO_TRACE_ROWS_32                                                                          \
    AO_TRACE_ROW(0, 1) AO_TRACE_ROW(1, 2) AO_TRACE_ROW(2, 3) AO_TRACE_ROW(3, 4)                   \
    AO_TRACE_ROW(4, 5) AO_TRACE_ROW(5, 6) AO_TRACE_ROW(6, 7) AO_TRACE_ROW(7, 8)                   \
    AO_TRACE_ROW(8, 9) AO_TRACE_ROW(9, 10) AO_TRACE_ROW(10, 11) AO_TRACE_ROW(11, 12)              \
    AO_TRACE_ROW(12, 13) AO_TRACE_ROW(13, 14) AO_TRACE_ROW(14, 15) AO_TRACE_ROW(15, 16)           \
    AO_TRACE_ROW(16, 17) AO_TRACE_ROW(17, 18) AO_TRACE_ROW(18, 19) AO_TRACE_ROW(19, 20)           \
    AO_TRACE_ROW(20, 21) AO_TRACE_ROW(21, 22) AO_TRACE_ROW(22, 23) AO_TRACE_ROW(23, 24)           \
    AO_TRACE_ROW(24, 25) AO_TRACE_ROW(25, 26) AO_TRACE_ROW(26, 27) AO_TRACE_ROW(27, 28)           \
    AO_TRACE_ROW(28, 29) AO_TRACE_ROW(29, 30) AO_TRACE_ROW(30, 31) AO_TRACE_ROW(31, 32)

// Ray-trace one tile: rows ifirst .. ifirst+31, columns jfirst + {tid, tid + NT} of source `sp` at time step
// `step`.  acc[i] receives the packed (column tid, column tid+NT) layer sums MINUS the piston references;
// refsum[c] their FP64 sum over the layers.  GROUP = number of adjacent lanes that share one reference
// (power of two <= 32; the n threads of a subaperture in k_fused, 1 in k_trace_tiled).
// `tiles` is the dynamic shared memory ([ns][rows][pitch] floats, 128-byte aligned).  All NT threads call it.
// On return every thread has finished reading the stages, but other warps may not have: __syncthreads()
// before reusing the memory.
template <int NT, int GROUP>
__device__ __forceinline__ void trace_tile(const TraceArgs& A, const SourceP& sp, TraceShared& S, float* tiles,
                                           const int jfirst, const int ifirst, const long long step,
                                           u64 (&acc)[kTraceRows], double (&refsum)[2])
{
    constexpr int NR = kTraceRows, NCOL = 2 * NT;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int pitch = A.pitch, ns = A.ns;
    const int tile_floats = A.rows * pitch;

    // ---- per-CTA layer table (FP64): column origin/increment, row origin, staged box ----
    if (tid == 0) {
        int na = 0;
        for (int l = 0; l < A.n_layers; ++l)
            if (A.layers[l].height < sp.H) S.act[na++] = l;
        S.nact = na;
        for (int s = 0; s < kTraceMaxStages; ++s) { mbar_init(&S.full_bar[s], 1); mbar_init(&S.empty_bar[s], NT / 32); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    {
        const double t = (double)step * A.dt;
        for (int l = tid; l < A.n_layers; l += NT) {
            const LayerP lp = A.layers[l];
            const double gamma = 1.0 - lp.height * sp.inv_H;
            const double x0 = -0.5 * (double)(sp.N - 1) * sp.d;
            const double c = 0.5 * (double)(lp.S - 1);
            double du = gamma * sp.d * lp.inv_pitch;
            if (fabs(du - 1.0) < 1e-9) du = 1.0;                     // same-pitch grids: exactly one pixel per sample
            const double u0 = (gamma * x0 + lp.height * sp.thx - lp.wx * t) * lp.inv_pitch + c;
            const double v0 = (gamma * x0 + lp.height * sp.thy - lp.wy * t) * lp.inv_pitch + c;
            const double vrow0 = fma((double)ifirst, du, v0);        // row coordinate of tile row 0
            const double ufirst = fma((double)jfirst, du, u0);
            const long long c0 = (long long)floor(ufirst) & ~3LL;    // 16-byte aligned start column
            const long long clast = (long long)floor(fma((double)(NCOL - 1), du, ufirst)) + 2;
            const long long rlast = (long long)floor(fma((double)(NR - 1), du, vrow0)) + 2;
            int wt = (int)(clast - c0 + 1); wt = (wt + 3) & ~3; if (wt > pitch) wt = pitch;
            int rt = (int)(rlast - (long long)floor(vrow0) + 1); if (rt > A.rows - 1) rt = A.rows - 1;
            S.u0[l] = u0; S.du[l] = du; S.v0[l] = vrow0; S.c0[l] = (double)c0; S.wt[l] = wt; S.rt[l] = rt;
        }
    }
    __syncthreads();
    const int nact = S.nact;

    // producer (warp 0): row schedule + TMA bulk row copies of active layer `a` into `stage`
    auto issue = [&](int a, int stage) {
        const int l = S.act[a];
        const LayerP lp = A.layers[l];
        const int wt = S.wt[l], rt = S.rt[l];
        const long long c0 = (long long)S.c0[l];
        const double vrow0 = S.v0[l], du = S.du[l];
        const long long r0 = (long long)floor(vrow0);
        {
            const double v = fma((double)lane, du, vrow0);
            const double vfl = floor(v);
            const float fy = fminf((float)(v - vfl), 0x1.fffffep-1f);
            const int r = (int)((long long)vfl - r0);
            const int rprev = __shfl_up_sync(0xffffffffu, r, 1);
            const int adv = (lane > 0 && r != rprev) ? 1 : 0;
            S.sched[stage][lane] = make_float4(1.0f - fy, fy, __int_as_float(adv), 0.0f);
        }
        uint64_t* bar = &S.full_bar[stage];
        float* dst = tiles + (size_t)stage * tile_floats;
        __syncwarp();
        if (lane == 0) mbar_expect_tx(bar, (uint32_t)(rt * wt) * 4u);
        __syncwarp();
        long long cw = c0 % lp.S; if (cw < 0) cw += lp.S;
        const int first = (cw + wt <= lp.S) ? wt : (int)(lp.S - cw);          // floats before the periodic wrap
        for (int r = lane; r < rt; r += 32) {
            long long rr = (r0 + r) % lp.S; if (rr < 0) rr += lp.S;
            const float* srow = lp.screen + (size_t)rr * lp.S;
            bulk_g2s(dst + r * pitch, srow + cw, (uint32_t)first * 4u, bar);
            if (first < wt) bulk_g2s(dst + r * pitch + first, srow, (uint32_t)(wt - first) * 4u, bar);
        }
    };
    if (warp == 0)
        for (int a = 0; a < ns && a < nact; ++a) issue(a, a);

#pragma unroll
    for (int i = 0; i < NR; ++i) acc[i] = 0ull;
    refsum[0] = 0.0; refsum[1] = 0.0;

    // column coordinates of this thread's two columns for layer ordinal `a` (FP64, one layer ahead of use)
    struct ColCoord { int jrel[2]; float fx[2]; };
    auto coords = [&](int a) {
        ColCoord cc;
        const int l = S.act[a];
        const double du = S.du[l], u0 = S.u0[l], c0d = S.c0[l];
#pragma unroll
        for (int c = 0; c < 2; ++c) {
            const double u = fma((double)(jfirst + c * NT + tid), du, u0);
            const double uf = floor(u);
            cc.fx[c] = fminf((float)(u - uf), 0x1.fffffep-1f);
            cc.jrel[c] = (int)(uf - c0d);
        }
        return cc;
    };
    ColCoord cur = {};
    if (nact > 0) cur = coords(0);
    const uint32_t tiles_s = smem_u32(tiles);
    const uint32_t pb = (uint32_t)pitch * 4u;

    int stage = 0, pstage = 0;
    uint32_t par = 0, ppar = 0;                // stage/parity of layer a and of layer a-1
    for (int a = 0; a < nact; ++a) {
        ColCoord nxt = cur;
        if (a + 1 < nact) nxt = coords(a + 1);
        // refill the stage that layer a-1 used, once every warp has released it
        if (warp == 0 && a >= 1 && a - 1 + ns < nact) {
            mbar_wait(&S.empty_bar[pstage], ppar);
            issue(a - 1 + ns, pstage);
        }
        mbar_wait(&S.full_bar[stage], par);
        const float* tile = tiles + (size_t)stage * tile_floats;
        const uint32_t tile_s = tiles_s + (uint32_t)stage * (uint32_t)tile_floats * 4u;
        float r0f, r1f;
        {
            const int j0 = __shfl_sync(0xffffffffu, cur.jrel[0], lane & ~(GROUP - 1));
            const int j1 = __shfl_sync(0xffffffffu, cur.jrel[1], lane & ~(GROUP - 1));
            r0f = tile[j0]; r1f = tile[j1];
        }
        refsum[0] += (double)r0f; refsum[1] += (double)r1f;
        const u64 ref = pack2(r0f, r1f), fx = pack2(cur.fx[0], cur.fx[1]);
        const float* ta = tile + cur.jrel[0];
        const float* tb = tile + cur.jrel[1];
        u64 Xa, Xb, p0, p1;
        {
            const u64 s0 = pack2(ta[0], tb[0]), s1 = pack2(ta[1], tb[1]);
            Xa = fma2(fx, sub2(s1, s0), sub2(s0, ref));
            const u64 s2 = pack2(ta[pitch], tb[pitch]), s3 = pack2(ta[pitch + 1], tb[pitch + 1]);
            Xb = fma2(fx, sub2(s3, s2), sub2(s2, ref));
            p0 = pack2(ta[2 * pitch], tb[2 * pitch]);
            p1 = pack2(ta[2 * pitch + 1], tb[2 * pitch + 1]);
        }
        uint32_t tp0 = tile_s + (uint32_t)(cur.jrel[0] + 2 * pitch) * 4u;
        uint32_t tp1 = tile_s + (uint32_t)(cur.jrel[1] + 2 * pitch) * 4u;
        const float4* sch = S.sched[stage];
        goto LE_0;
        AO_TRACE_ROWS_32
        LE_32: LO_32: ;
        cur = nxt;
        __syncwarp();
        if (lane == 0) mbar_arrive(&S.empty_bar[stage]);
        pstage = stage; ppar = par;
        if (++stage == ns) { stage = 0; par ^= 1u; }
    }
}

}  // namespace ao
