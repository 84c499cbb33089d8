// trace2.cuh -- tiled ray-trace core of k_fused: one CTA traces a tile of 16 output rows x 2 NT output
// columns of one source for TWO consecutive time steps.  PAPER.md:56 (frozen flow), PAPER.md:60 (open-loop
// wavefront of every star, finite-distance projection of the LGS); reading O2 of DESIGN.md section 3.
//
// Why two steps per CTA: under frozen flow the footprints of steps k and k+1 differ by a sub-pixel to
// few-pixel wind shift, so one staged screen box (the union of both footprints) serves both; that halves the
// L2 -> shared-memory traffic per traced sample and keeps a stage small enough for three stages in flight at
// four CTAs per SM.
//
// Per layer the box is staged by TMA bulk row copies issued by warp 0 (full/empty mbarrier pipeline, no
// CTA-wide barrier in the layer loop).  Each thread owns two columns (tid, tid + NT) packed in one 64-bit
// register pair so that the inner loop is FFMA2 / FADD2.  Bilinear interpolation is separable: an output row
// combines x-interpolated screen rows with warp-uniform y-weights.  Warp 0 writes, with each stage it issues,
// the row table of that (layer, two steps), built in 32.32 fixed point: per output row the weights and the shared-memory offset of its
// bottom screen row, so the row march (t2_march) is branch-free straight-line code.
// Column coordinates are 32.32 fixed point: cell and fraction of column j are the two halves of
// uf + j * du (one IMAD.WIDE), exact to 2^-32 pixel at any screen coordinate.
// Precision: a warp-uniform piston reference (a tap of the box) is subtracted from every tap so that the fp32
// sums stay at the few-radian level (|FFT|^2 is piston-invariant per subaperture; a warp never splits one).
#pragma once
#include "ao_device.cuh"
#include "pk_tma.cuh"

#include <type_traits>

namespace ao {

template <int I, int N, typename F>
__device__ __forceinline__ void static_for_t2(F&& f)
{
    if constexpr (I < N) {
        f(std::integral_constant<int, I>{});
        static_for_t2<I + 1, N>(static_cast<F&&>(f));
    }
}

constexpr int kTR = 16;                 // output rows of a tile
constexpr int kKS = 2;                  // time steps per CTA
constexpr int kT2MaxStages = 4;

struct Trace2Args {
    const LayerP* layers; int n_layers;
    const SourceP* srcs;
    long long step0; double dt;
    int pitch;            // staged row pitch in floats (multiple of 4)
    int rows;             // staged rows allocated per stage (box rows + 1 prefetch pad row)
    int ns;               // stages in flight
    const unsigned char* tmaps;   // per-layer CUtensorMap[n_layers] (128 bytes each), then int2 box {pitch_l, rows_l}[n_layers]; or NULL
#ifdef AO_PROFILE_SWITCHES
    int dbg;              // profiling builds only (AO_DBG): 1 = skip the row march, 2 = skip staging, 4 = skip image formation
#endif
};

// Component-timing switches exist in profiling builds only (AO_BUILD_PROFILE=1); a normal build compiles them out.
#ifdef AO_PROFILE_SWITCHES
#define AO_DBG_ON(args, bit) (((args).dbg & (bit)) != 0)
#else
#define AO_DBG_ON(args, bit) false
#endif

// Per active layer, built in the prologue (dynamic shared memory).
struct __align__(16) LayerT {
    const float* scr;     // screen base
    int S;                // screen side
    int cw, rw;           // start column / row of the staged box, wrapped into [0, S)
    int wt, rt;           // box width (multiple of 4) and rows
    unsigned duf;         // frac(du) 2^32
    int du_hi;            // floor(du)
    int lay;              // layer index
    int tm;               // 1: the box does not wrap the screen edge and a tensor map exists: one TMA tensor copy
    int pitch, box_rows;  // shared-memory row pitch of this layer's box (the map's own box with a tensor copy) and its rows
    double du;            // screen pixels per output sample
    u64 vf[kKS];          // (row coordinate of tile row 0 - box row 0) 2^32
    u64 uf[kKS];          // (column coordinate of tile column 0 - box column 0) 2^32
};
// Unit march (du = 1): vf / uf are replaced, in place, by what its consumers need: the box row of the top tap of tile
// row 0 and the box column of tile column 0 (per step), and the two fractional weights of the whole tile.
struct UnitT { float fy[kKS], fx[kKS]; int row[kKS], col[kKS]; };
static_assert(sizeof(UnitT) == sizeof(u64) * kKS + sizeof(u64) * kKS, "UnitT overlays LayerT::vf and LayerT::uf");
__device__ __forceinline__ UnitT* unit_of(LayerT& T) { return reinterpret_cast<UnitT*>(&T.vf[0]); }
__device__ __forceinline__ const UnitT* unit_of(const LayerT& T) { return reinterpret_cast<const UnitT*>(&T.vf[0]); }

struct __align__(16) Trace2Shared {
    uint64_t full_bar[kT2MaxStages], empty_bar[kT2MaxStages];
    int nact;
};

__host__ __device__ inline size_t trace2_sched_bytes(int n_layers)
{
    return (size_t)n_layers * sizeof(LayerT) + (sizeof(float4) * kTR + sizeof(int) * 8) * kKS * kT2MaxStages;
}

// ---- the 16 output rows of one (layer, step): straight-line row march ----
// Output row i interpolates between the x-interpolated screen rows X[r_i] (top) and X[r_i + 1] (bottom).
// Every row builds ITS OWN bottom row N_i = X[r_i + 1] from four taps at a table-driven shared-memory offset
// (no carried pointer, no condition).  Because 1/2 <= du <= 1, consecutive output rows advance by 0 or 1 screen
// rows and never stall twice in a row, so the top row is N_{i-1} (advance) or N_{i-2} (no advance): the
// prologue folds that choice into the weights, acc_i += w1 N_i + a N_{i-1} + b N_{i-2} with (a, b) =
// (w0, 0) or (0, w0).  The march is therefore one basic block with static registers: no branch (a taken
// branch per row starved the instruction fetch), no select, and every row's loads are independent of the
// previous rows', so ptxas overlaps the shared-memory latency of one row with the FFMA2 chains of others.
// Table entry of row i (16 bytes): (w1, a, b, byte offset of X[r_i + 1] relative to X[r_0]).
__device__ __forceinline__ u64 t2_xrow(const uint32_t a0, const uint32_t a1, const u64 fx, const u64 ref)
{
    const u64 p0 = pack2(lds_f32(a0), lds_f32(a1));
    const u64 p1 = pack2(lds_f32_next(a0), lds_f32_next(a1));
    return fma2(fx, sub2(p1, p0), sub2(p0, ref));
}

// acc[OFF .. OFF+15] += the layer's contribution for one step.  tp0 / tp1: shared-memory byte addresses of the
// left tap of the thread's two columns in box row r_0 (top tap of output row 0); wtab: shared-memory byte
// address of the 16 table entries.
template <int OFF>
__device__ __forceinline__ void t2_march(u64 (&acc)[kKS * kTR], const uint32_t tp0, const uint32_t tp1,
                                         const u64 fx, const u64 ref, const uint32_t wtab)
{
    u64 n1 = t2_xrow(tp0, tp1, fx, ref), n2 = n1;
#pragma unroll
    for (int i = 0; i < kTR; ++i) {
        const float4 w = lds_f32x4(wtab + 16u * (uint32_t)i);
        const uint32_t off = __float_as_uint(w.w);
        const u64 n0 = t2_xrow(tp0 + off, tp1 + off, fx, ref);
        acc[OFF + i] = fma2(pack2(w.x, w.x), n0, fma2(pack2(w.y, w.y), n1, fma2(pack2(w.z, w.z), n2, acc[OFF + i])));
        n2 = n1; n1 = n0;
    }
}

// The same for ANY du > 0 (screen pixels per output sample): acc_i += w0 X[r_i] + w1 X[r_i + 1].  Every output row builds
// its bottom x-interpolated row from four taps; its top row is the previous row's bottom row when the march advanced by
// exactly one screen row (for 1 <= du < 2 that is a fraction 2 - du of the rows), otherwise it is built from four more
// taps, loaded under a warp-uniform predicate (predicated-off loads cost an issue slot, no shared-memory wavefront: at
// du > 1 every tap load is two wavefronts, which is what bounds c4 at M = 16).  Still one basic block.  Used when a layer
// falls outside 1/2 <= du <= 1 (c4 at M = 16: the WFS grid is coarser than the screens, du up to 1.5; low beacons).
// Table entry: (w0, w1, byte offset of X[r_i] relative to X[r_0], flag: 1 = build the top row).
template <int OFF>
__device__ __forceinline__ void t2_march_any(u64 (&acc)[kKS * kTR], const uint32_t tp0, const uint32_t tp1, const uint32_t pb,
                                             const u64 fx, const u64 ref, const uint32_t wtab)
{
    u64 prev = 0ull;
#pragma unroll
    for (int i = 0; i < kTR; ++i) {
        const float4 w = lds_f32x4(wtab + 16u * (uint32_t)i);
        const uint32_t off = __float_as_uint(w.z), flag = __float_as_uint(w.w);
        const u64 bot = t2_xrow(tp0 + off + pb, tp1 + off + pb, fx, ref);
        float a0, a1, b0, b1;
        lds_f32_pair_if(tp0 + off, flag, a0, a1);
        lds_f32_pair_if(tp1 + off, flag, b0, b1);
        const u64 p0 = pack2(a0, b0), p1 = pack2(a1, b1);
        const u64 built = fma2(fx, sub2(p1, p0), sub2(p0, ref));
        const u64 top = flag ? built : prev;
        acc[OFF + i] = fma2(pack2(w.y, w.y), bot, fma2(pack2(w.x, w.x), top, acc[OFF + i]));
        prev = bot;
    }
}

// For du <= 2/3 (fine WFS grids: c4 at M = 64 has du ~ 0.3): four consecutive output rows lie within three
// screen-row intervals, so a group of four rows builds four x-interpolated rows X[r_g .. r_g + 3] once (4 tap loads
// per output row, as in t2_march) and every row is a four-weight combination of them (two weights non-zero).
// Table entry of row i: its four weights; gtab: the byte offsets of the four groups' first row relative to X[r_0].
template <int OFF>
__device__ __forceinline__ void t2_march_quad(u64 (&acc)[kKS * kTR], const uint32_t tp0, const uint32_t tp1, const uint32_t pb,
                                              const u64 fx, const u64 ref, const uint32_t wtab, const uint32_t gtab)
{
    const float4 go = lds_f32x4(gtab);
    const uint32_t goff[4] = {__float_as_uint(go.x), __float_as_uint(go.y), __float_as_uint(go.z), __float_as_uint(go.w)};
#pragma unroll
    for (int g = 0; g < 4; ++g) {
        const uint32_t a0 = tp0 + goff[g], a1 = tp1 + goff[g];
        const u64 x0 = t2_xrow(a0, a1, fx, ref), x1 = t2_xrow(a0 + pb, a1 + pb, fx, ref);
        const u64 x2 = t2_xrow(a0 + 2 * pb, a1 + 2 * pb, fx, ref), x3 = t2_xrow(a0 + 3 * pb, a1 + 3 * pb, fx, ref);
#pragma unroll
        for (int i = 4 * g; i < 4 * g + 4; ++i) {
            const float4 w = lds_f32x4(wtab + 16u * (uint32_t)i);
            acc[OFF + i] = fma2(pack2(w.w, w.w), x3, fma2(pack2(w.z, w.z), x2, fma2(pack2(w.y, w.y), x1,
                           fma2(pack2(w.x, w.x), x0, acc[OFF + i]))));
        }
    }
}

// du == 1 exactly (grids with the screen pitch seen from infinity: the NGS sensors and the science directions): every
// output row advances by one screen row and every column by one cell, so the bilinear weights are the same for the
// whole tile and the box rows are consecutive: no table, and with the compile-time row pitch kUnitPitch every tap load
// has an immediate offset.  acc_i += w0 X[r_0 + i] + w1 X[r_0 + i + 1].
constexpr int kUnitPitch = 272;         // floats: 256 columns + wind shift of the paired step + alignment slack
template <int ROW>
__device__ __forceinline__ u64 t2_xrow_unit(const uint32_t a0, const uint32_t a1, const u64 fx, const u64 ref)
{
    constexpr int O = ROW * kUnitPitch * 4;
    const u64 p0 = pack2(lds_f32_imm<O>(a0), lds_f32_imm<O>(a1));
    const u64 p1 = pack2(lds_f32_imm<O + 4>(a0), lds_f32_imm<O + 4>(a1));
    return fma2(fx, sub2(p1, p0), sub2(p0, ref));
}
template <int OFF>
__device__ __forceinline__ void t2_march_unit(u64 (&acc)[kKS * kTR], const uint32_t tp0, const uint32_t tp1, const u64 fx,
                                              const u64 ref, const float w0, const float w1)
{
    const u64 W0 = pack2(w0, w0), W1 = pack2(w1, w1);
    u64 prev = t2_xrow_unit<0>(tp0, tp1, fx, ref);
    static_for_t2<0, kTR>([&](auto ii) {
        constexpr int i = decltype(ii)::value;
        const u64 cur = t2_xrow_unit<i + 1>(tp0, tp1, fx, ref);
        acc[OFF + i] = fma2(W1, cur, fma2(W0, prev, acc[OFF + i]));
        prev = cur;
    });
}

// Ray-trace one tile for two steps: rows ifirst .. ifirst+15, columns jfirst + {tid, tid + NT} of source `sp` at
// time steps step_first and step_first + 1.  acc[s * 16 + i] receives the packed (column tid, column tid + NT)
// layer sums of step s, row i, minus warp-uniform piston references (the same for both steps); with REFSUM
// their FP64 sums over the layers are returned in refsum[column] so that callers can restore absolute phase.
// `dyn`: dynamic shared memory, 128-byte aligned: [ns][rows][pitch] floats, then trace2_sched_bytes(n_layers).
// All NT threads call it.  On return every thread has finished reading the stages, but other warps may not
// have: __syncthreads() before reusing the memory.
// PARTIAL: the tile is narrower than 2 NT columns (a work item with fewer subapertures than the tile holds): the thread's
// second column is tid + pair_off instead of tid + NT (pair_off a multiple of 32, at most NT), so the first pair_off
// threads cover columns 0 .. 2 pair_off - 1 and the warps from pair_off on skip the row marches (their acc stays zero);
// they still take their producer turns and barrier arrivals.
template <int NT, bool REFSUM, int MODE, bool PARTIAL = false>
__device__ __forceinline__ void trace2_tile(const Trace2Args& A, const SourceP& sp, Trace2Shared& S, unsigned char* dyn,
                                            const int jfirst, const int ifirst, const long long step_first,
                                            u64 (&acc)[kKS * kTR], double (&refsum)[2], const int pair_off = NT)
{
    constexpr int NCOL = 2 * NT;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int PO = PARTIAL ? pair_off : NT;                  // column distance of the thread's packed pair
    const bool idle = PARTIAL && tid >= PO;
    const int pitch = A.pitch, ns = A.ns;
    const int tile_floats = A.rows * pitch;
    float* tiles = reinterpret_cast<float*>(dyn);
    LayerT* L = reinterpret_cast<LayerT*>(dyn + (size_t)ns * tile_floats * sizeof(float));
    float4* Wt = reinterpret_cast<float4*>(L + A.n_layers);       // [stage][step][row] table entries
    int* R0 = reinterpret_cast<int*>(Wt + kT2MaxStages * kKS * kTR);   // [stage][step] box row of the top tap of row 0
    int* G = R0 + 4 * kKS * kT2MaxStages;                              // [stage][step][4] group offsets of the quad march

    if (tid == 0) {
        int na = 0;
        for (int l = 0; l < A.n_layers; ++l)
            if (A.layers[l].height < sp.H) L[na++].lay = l;
        S.nact = na;
        for (int s = 0; s < kT2MaxStages; ++s) { mbar_init(&S.full_bar[s], 1); mbar_init(&S.empty_bar[s], NT / 32); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const int nact = S.nact;

    // ---- per-layer geometry (FP64): staged box = union of the footprints of both steps ----
    for (int a = tid; a < nact; a += NT) {
        LayerT& T = L[a];
        const LayerP lp = A.layers[T.lay];
        const double gamma = 1.0 - lp.height * sp.inv_H;
        const double x0 = -0.5 * (double)(sp.N - 1) * sp.d;
        const double c = 0.5 * (double)(lp.S - 1);
        double du = gamma * sp.d * lp.inv_pitch;
        if (fabs(du - 1.0) < 1e-9) du = 1.0;                     // same-pitch grids: exactly one pixel per sample
        double uf[kKS], vf[kKS];
        long long cmin = 0, cmax = 0, rmin = 0, rmax = 0;
#pragma unroll
        for (int s = 0; s < kKS; ++s) {
            const double t = (double)(step_first + s) * A.dt;
            const double u0 = (gamma * x0 + lp.height * sp.thx - lp.wx * t) * lp.inv_pitch + c;
            const double v0 = (gamma * x0 + lp.height * sp.thy - lp.wy * t) * lp.inv_pitch + c;
            uf[s] = fma((double)jfirst, du, u0);
            vf[s] = fma((double)ifirst, du, v0);
            const long long c_lo = (long long)floor(uf[s]) & ~3LL;                         // 16-byte aligned start
            const long long c_hi = (long long)floor(fma((double)(NCOL - 1), du, uf[s])) + 2;
            const long long r_lo = (long long)floor(vf[s]);
            // 2^-20: the row table is built in 32.32 fixed point and may land one row further than the FP64 floor
            long long r_hi = (long long)floor(fma((double)(kTR - 1), du, vf[s]) + 9.5367431640625e-7) + 1;
            if (MODE == 2) r_hi = max(r_hi, (long long)floor(fma((double)(kTR - 4), du, vf[s]) + 9.5367431640625e-7) + 3);   // last group's fourth row
            if (s == 0 || c_lo < cmin) cmin = c_lo;
            if (s == 0 || c_hi > cmax) cmax = c_hi;
            if (s == 0 || r_lo < rmin) rmin = r_lo;
            if (s == 0 || r_hi > rmax) rmax = r_hi;
        }
        int wt = (int)(cmax - cmin + 1); wt = (wt + 3) & ~3; if (wt > pitch) wt = pitch;
        int rt = (int)(rmax - rmin + 1); if (rt > A.rows - 1) rt = A.rows - 1;
        long long cw = cmin % lp.S; if (cw < 0) cw += lp.S;
        long long rw = rmin % lp.S; if (rw < 0) rw += lp.S;
        T.scr = lp.screen; T.S = lp.S; T.cw = (int)cw; T.rw = (int)rw; T.wt = wt; T.rt = rt;
        T.tm = 0; T.pitch = pitch; T.box_rows = 0;
        if (A.tmaps != nullptr) {                                  // this layer's own box {pitch_l, rows_l}: no overfetch
            const int2 bx = reinterpret_cast<const int2*>(A.tmaps + (size_t)A.n_layers * 128)[T.lay];
            if (wt <= bx.x && rt <= bx.y && cw + wt <= lp.S && rw + rt <= lp.S) { T.tm = 1; T.pitch = bx.x; T.box_rows = bx.y; }
        }
        T.du = du; T.du_hi = (int)floor(du);
        const unsigned long long f = __double2ull_rn((du - (double)T.du_hi) * 4294967296.0);
        T.duf = f > 0xffffffffull ? 0xffffffffu : (unsigned)f;
        if (MODE == 3) {                                           // du = 1: one cell offset and one weight pair per step
            UnitT u;
#pragma unroll
            for (int s = 0; s < kKS; ++s) {
                const double ur = uf[s] - (double)cmin, vr = vf[s] - (double)rmin, fu = floor(ur), fv = floor(vr);
                u.col[s] = (int)fu; u.fx[s] = (float)(ur - fu);
                u.row[s] = (int)fv; u.fy[s] = (float)(vr - fv);
            }
            *unit_of(T) = u;
        } else {
#pragma unroll
            for (int s = 0; s < kKS; ++s) {
                T.uf[s] = __double2ull_rn((uf[s] - (double)cmin) * 4294967296.0);
                T.vf[s] = __double2ull_rn((vf[s] - (double)rmin) * 4294967296.0);
            }
        }
    }
    __syncthreads();

    // producer (one warp): row table + TMA bulk row copies of active layer `a` into `stage`
    auto issue = [&](int a, int stage) {
        const LayerT& T = L[a];
        const int wt = T.wt, rt = T.rt, Sn = T.S, cw = T.cw, rw = T.rw, pitch = T.pitch;
        const float* scr = T.scr;
        uint64_t* bar = &S.full_bar[stage];
        float* dst = tiles + (size_t)stage * tile_floats;
        if (MODE != 3) {   // row table of this stage: lane = step * 16 + row; the unit march needs none
            static_assert(kKS * kTR == 32, "one lane per (step, row)");
            // Row coordinates in 32.32 fixed point like the columns: row and fraction of tile row i are the two halves of
            // vf + i du, exact to 2^-32 pixel per added du (the FP64 form of this table, floor and int <-> double conversions
            // of 64-bit values, was 8 % of k_fused's stall samples: one warp per layer computes it inside the layer loop).
            const int s = lane / kTR, i = lane - s * kTR;
            const u64 du64t = ((u64)(unsigned)T.du_hi << 32) | (u64)T.duf;
            const u64 V = T.vf[s] + (u64)(unsigned)i * du64t;
            int r = (int)(V >> 32);
            float fy = __uint2float_rn((unsigned)V) * 2.3283064365386963e-10f;            // may round to 1: same value by continuity
            if (r + 1 >= T.rt) { r = T.rt - 2; fy = 1.0f; }                                // never a tap beyond the staged box
            const int rprev = __shfl_up_sync(0xffffffffu, r, 1);
            const int r0 = __shfl_sync(0xffffffffu, r, s * kTR);
            const bool adv = i == 0 || r != rprev;
            const float w0 = 1.0f - fy;
            if (MODE == 2) {
                // rows in groups of four share four x-interpolated screen rows starting at the group's first top row
                const int rg = __shfl_sync(0xffffffffu, r, lane & ~3);
                const int j = r - rg;                                            // 0 .. 2 for du <= 2/3
                const float c0 = w0, c1 = fy;
                Wt[stage * (kKS * kTR) + lane] = make_float4(j == 0 ? c0 : 0.0f, j == 0 ? c1 : (j == 1 ? c0 : 0.0f),
                                                              j == 1 ? c1 : (j == 2 ? c0 : 0.0f), j == 2 ? c1 : 0.0f);
                if ((i & 3) == 0) G[(stage * kKS + s) * 4 + (i >> 2)] = (r - r0) * pitch * 4;
            } else if (MODE == 1) {
                const uint32_t build_top = (i == 0 || r != rprev + 1) ? 1u : 0u;   // else the top row is the previous bottom row
                Wt[stage * (kKS * kTR) + lane] = make_float4(w0, fy, __uint_as_float((uint32_t)((r - r0) * pitch * 4)),
                                                              __uint_as_float(build_top));
            } else
            Wt[stage * (kKS * kTR) + lane] = make_float4(fy, adv ? w0 : 0.0f, adv ? 0.0f : w0,
                                                          __uint_as_float((uint32_t)((r + 1 - r0) * pitch * 4)));
            if (i == 0) R0[stage * kKS + s] = r;
        }
        __syncwarp();
        if (AO_DBG_ON(A, 2)) return;
        if (T.tm) {                                        // whole box in one tensor copy (rows beyond the screen: zero fill)
            if (lane == 0) {
                mbar_expect_tx(bar, (uint32_t)(T.pitch * T.box_rows) * 4u);
                tma_load_2d(dst, A.tmaps + (size_t)T.lay * 128, cw, rw, bar);
            }
            return;
        }
        if (lane == 0) mbar_expect_tx(bar, (uint32_t)(rt * wt) * 4u);
        __syncwarp();
        const int first = (cw + wt <= Sn) ? wt : Sn - cw;                     // floats before the periodic wrap
        for (int r = lane; r < rt; r += 32) {
            int rr = rw + r; if (rr >= Sn) rr -= Sn;
            const float* srow = scr + (size_t)rr * Sn;
            bulk_g2s(dst + r * pitch, srow + cw, (uint32_t)first * 4u, bar);
            if (first < wt) bulk_g2s(dst + r * pitch + first, srow, (uint32_t)(wt - first) * 4u, bar);
        }
    };
    if (warp == 0)
        for (int a = 0; a < ns && a < nact; ++a) issue(a, a);

#pragma unroll
    for (int i = 0; i < kKS * kTR; ++i) acc[i] = 0ull;
    refsum[0] = 0.0; refsum[1] = 0.0;
    __syncthreads();

    const uint32_t tiles_s = smem_u32(tiles), w_s = smem_u32(Wt);
    const uint32_t tile_bytes = (uint32_t)tile_floats * 4u;
    int stage = 0;
    uint32_t par = 0;                          // stage and parity of layer a
    // Refill lag: at iteration a the producer refills the stage of layer a - lag with layer a - lag + ns.  With
    // lag = 1 it would wait for the slowest warp to finish the layer it has just finished itself (a CTA-wide
    // rendezvous every layer, measured as 22 % of all stall samples); with lag = 2 the stage being recycled was
    // released a whole layer ago and the copy still has one full layer of compute to land.
    const int lag = ns >= 3 ? 2 : 1;
    for (int a = 0; a < nact; ++a) {
        // the producer role rotates over the warps: a fixed producer warp would lag by its issue + table time
        // every layer and pace the whole CTA
        if (warp == (a & (NT / 32 - 1)) && a >= lag && a - lag + ns < nact && !AO_DBG_ON(A, 8)) {
            const int l = a - lag, m = l / ns;
            mbar_wait(&S.empty_bar[l - m * ns], (uint32_t)(m & 1));
            issue(l + ns, l - m * ns);
        }
        const LayerT& T = L[a];
        if (MODE == 3) {
            // du = 1: every per-thread quantity is the layer's (row, column, fx, fy) plus the thread's column index
            const uint32_t tile_u = tiles_s + (uint32_t)stage * tile_bytes;
            if (!AO_DBG_ON(A, 2)) mbar_wait(&S.full_bar[stage], par);
            const UnitT u = *unit_of(T);
            const uint32_t b0 = tile_u + ((uint32_t)u.row[0] * kUnitPitch + (uint32_t)u.col[0]) * 4u;
            const uint32_t b1 = tile_u + ((uint32_t)u.row[1] * kUnitPitch + (uint32_t)u.col[1]) * 4u;
            const float r0f = lds_f32(b0 + (uint32_t)(tid & ~31) * 4u), r1f = lds_f32(b0 + (uint32_t)((tid & ~31) + PO) * 4u);
            const u64 ref = pack2(r0f, r1f);
            if (REFSUM) { refsum[0] += (double)r0f; refsum[1] += (double)r1f; }
            if (!AO_DBG_ON(A, 1) && !idle) {
                t2_march_unit<0>(acc, b0 + (uint32_t)tid * 4u, b0 + (uint32_t)(tid + PO) * 4u, pack2(u.fx[0], u.fx[0]), ref, 1.0f - u.fy[0], u.fy[0]);
                t2_march_unit<kTR>(acc, b1 + (uint32_t)tid * 4u, b1 + (uint32_t)(tid + PO) * 4u, pack2(u.fx[1], u.fx[1]), ref, 1.0f - u.fy[1], u.fy[1]);
            }
        } else {
        const uint32_t pb = (uint32_t)T.pitch * 4u;
        const u64 du64 = ((u64)(unsigned)T.du_hi << 32) | (u64)T.duf;
        const u64 uf0 = T.uf[0], uf1 = T.uf[1];
        const uint32_t tile_s = tiles_s + (uint32_t)stage * tile_bytes;
        const u64 colA = (u64)(unsigned)tid * du64, colB = colA + (u64)(unsigned)PO * du64;
        const u64 colW = (u64)(unsigned)(tid & ~31) * du64;
        if (!AO_DBG_ON(A, 2)) mbar_wait(&S.full_bar[stage], par);
        const int ro0 = R0[stage * kKS], ro1 = R0[stage * kKS + 1];
        u64 ref;
        {
            const u64 a0 = uf0 + colW, a1 = a0 + (u64)(unsigned)PO * du64;
            const uint32_t rowb = tile_s + (uint32_t)ro0 * pb;
            const float r0f = lds_f32(rowb + (uint32_t)(a0 >> 32) * 4u), r1f = lds_f32(rowb + (uint32_t)(a1 >> 32) * 4u);
            ref = pack2(r0f, r1f);
            if (REFSUM) { refsum[0] += (double)r0f; refsum[1] += (double)r1f; }
        }
        const float k32 = 2.3283064365386963e-10f;             // 2^-32
        if (!AO_DBG_ON(A, 1) && !idle) {
            {
                const u64 U0 = uf0 + colA, U1 = uf0 + colB;
                const u64 fx = pack2(__uint2float_rn((unsigned)U0) * k32, __uint2float_rn((unsigned)U1) * k32);
                const uint32_t rowb = tile_s + (uint32_t)ro0 * pb;
                const uint32_t t0 = rowb + (uint32_t)(U0 >> 32) * 4u, t1 = rowb + (uint32_t)(U1 >> 32) * 4u;
                const uint32_t wt_s = w_s + (uint32_t)(stage * kKS + 0) * (kTR * 16);
                if (MODE == 2) t2_march_quad<0>(acc, t0, t1, pb, fx, ref, wt_s, smem_u32(G + (stage * kKS + 0) * 4));
                else if (MODE == 1) t2_march_any<0>(acc, t0, t1, pb, fx, ref, wt_s);
                else t2_march<0>(acc, t0, t1, fx, ref, wt_s);
            }
            {
                const u64 U0 = uf1 + colA, U1 = uf1 + colB;
                const u64 fx = pack2(__uint2float_rn((unsigned)U0) * k32, __uint2float_rn((unsigned)U1) * k32);
                const uint32_t rowb = tile_s + (uint32_t)ro1 * pb;
                const uint32_t t0 = rowb + (uint32_t)(U0 >> 32) * 4u, t1 = rowb + (uint32_t)(U1 >> 32) * 4u;
                const uint32_t wt_s = w_s + (uint32_t)(stage * kKS + 1) * (kTR * 16);
                if (MODE == 2) t2_march_quad<kTR>(acc, t0, t1, pb, fx, ref, wt_s, smem_u32(G + (stage * kKS + 1) * 4));
                else if (MODE == 1) t2_march_any<kTR>(acc, t0, t1, pb, fx, ref, wt_s);
                else t2_march<kTR>(acc, t0, t1, fx, ref, wt_s);
            }
        }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&S.empty_bar[stage]);
        if (++stage == ns) { stage = 0; par ^= 1u; }
    }
}

}  // namespace ao
