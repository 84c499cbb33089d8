// k_fused.cu -- the WFS hot path: ray-trace + Shack-Hartmann image + centre of gravity in ONE kernel
// (ao_sh_images with phase_dev == NULL for M in {16, 32}, n = M/2, beta*P = M, P = 8; PAPER.md:56,60,28,82;
// readings O2, O3, O4, O5, O6).
//
// Work decomposition of k_fused.  A CTA (128 threads) processes one work item of one source for TWO
// consecutive time steps: a tile of 16 rows x 256 columns of phase samples = R2 = 16/n subaperture rows by up
// to G = 256/n horizontally adjacent subapertures, built at create time from runs of valid subapertures
// (invalid ones are never scheduled; their outputs are zero-filled by a memset).  The two steps share one
// staged screen box per layer (frozen flow: their footprints differ by the wind shift only).  CTAs of
// consecutive step pairs of the same tile are adjacent in the grid: all but the first hit in L2.
//
// Phase A, ray-trace: trace2.cuh.  The phase of the tile ends in registers; it never touches HBM.
//
// Phase B, image formation, one round per (subaperture row, column slot); the rounds are a rolled loop so
// that the FFT code exists once (instruction cache).  Thread (g, b) holds column b of subaperture g of the
// round: E[a] = A exp(i phi).  Column FFTs run entirely in registers: the half-pixel-centred, zero-padded
// M-point DFT of n inputs splits (first DIF stage on half-zero input) into two n-point FFTs of
// e[a] cis(pi (M-1) a/M) and e[a] cis(pi (M-3) a/M) with compile-time twiddles.  One transpose through
// padded shared memory (private to the n threads of the subaperture: __syncwarp only), then the row FFTs
// (two rows per thread), |.|^2, beta x beta binning (in-register over m, halving shuffles over k), optional
// noise, centre of gravity by warp shuffles.
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <type_traits>
#include <vector>

#include <cuda.h>
#include <cudaTypedefs.h>

#include "fft_reg.cuh"
#include "trace2.cuh"
#include "trace2_plan.cuh"

namespace ao {

struct WorkItem { int p, q0, cnt, pad; };

struct FusedArgs {
    Trace2Args T;
    const int* sel; int n_sel;
    const WorkItem* items; int n_items;
    int n_steps, n_pairs;
    const float* amp;                 // [N][N] on the WFS grid
    const uint8_t* valid;             // [n_sub^2]
    int n_sub;
    float norm;                       // 1/(M^2 n^2)
    NoiseP nz;
    float* images;                    // nullable [k][si][nsa][P][P]
    float* slopes;                    // nullable [k][si][2][nsa]
    SodiumP na;                       // extended beacon (ELONG kernels only; reading O9)
};


template <int M>
struct FusedCfg {
    static constexpr int n = M / 2;
    static constexpr int NT = kFusedThreads;
    static constexpr int R2 = kTR / n;                   // subaperture rows per tile
    static constexpr int G = kTileCols / n;              // subapertures per tile row
    static constexpr int GS = NT / n;                    // subapertures per round
    static constexpr int HS = kKS * R2;                  // (step, subaperture row) slices held in registers
    static constexpr int ROUNDS = 2 * HS;
    static constexpr int P = 8, BETA = M / 8;
    static constexpr int XP = n + 1;                     // transpose pitch (float2 units)
    static constexpr int SUB_STRIDE = M * XP + (n == 8 ? 8 : 0);
    static constexpr size_t XCH_BYTES = (size_t)GS * SUB_STRIDE * sizeof(float2);
    static_assert(kTR % n == 0 && NT % n == 0 && n <= 32, "bad fused configuration");
};

#ifndef AO_FUSED_MINB
#define AO_FUSED_MINB 3
#endif
template <int M, bool NOISE, bool ANYDU, bool MAPS, bool ELONG>
__global__ void __launch_bounds__(kFusedThreads, AO_FUSED_MINB)
k_fused(const FusedArgs A)
{
    using K = FusedCfg<M>;
    constexpr int n = K::n, NT = K::NT, R2 = K::R2, P = K::P, BETA = K::BETA;
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ Trace2Shared S;

    const int tid = threadIdx.x;
    // the step pair is the fastest block index: consecutive CTAs share their screen footprint through L2
    const int kp = (int)(blockIdx.x % (unsigned)A.n_pairs);
    const unsigned rest = blockIdx.x / (unsigned)A.n_pairs;
    const WorkItem it = A.items[rest % (unsigned)A.n_items];
    const int si = (int)(rest / (unsigned)A.n_items);
    const int src_index = A.sel[si];
    const SourceP sp = A.T.srcs[src_index];
    const int N = A.n_sub * n, nsa = A.n_sub * A.n_sub;

    // ---- phase A: ray-trace of the 16 x 256 tile, two steps, into registers ----
    u64 acc[kKS * kTR];
    double refsum[2];                                      // unused: |FFT|^2 is piston-invariant per subaperture
    // a narrow work item (a run's tail) packs its columns on the first warps: pair distance 32 / 64 / 128 columns
    // (not in the ELONG instantiations: one more live value there costs 56 bytes of spills in the scatterer loop)
    const int ncols = it.cnt * n;
    const int po = ELONG ? NT : (ncols > NT ? NT : (ncols > NT / 2 ? NT / 2 : NT / 4));
    trace2_tile<NT, false, ANYDU ? 1 : 0, !ELONG>(A.T, sp, S, smem, it.q0 * n, it.p * n, A.T.step0 + 2 * kp, acc, refsum, po);
    __syncthreads();                                       // stages are dead: shared memory becomes the exchange buffer

    // ---- phase B: image formation, one (subaperture row, column slot) round at a time ----
    float2* xch = reinterpret_cast<float2*>(smem);
    const float scale = (float)sp.scale;
    const float* mp = MAPS ? sp.map : nullptr;             // additive phase map of this source or NULL (ao_set_phase_map)
    const int g = tid / n, b = tid - g * n;                // subaperture in round, column in subaperture
    float2* xs = xch + (size_t)g * K::SUB_STRIDE;
#pragma unroll 1
    for (int rd = AO_DBG_ON(A.T, 4) ? K::ROUNDS : 0; rd < K::ROUNDS; ++rd) {
        const int hs = rd >> 1, c = rd & 1;                // hs = step-in-pair * R2 + subaperture row
        const int sp2 = hs / R2, h = hs - sp2 * R2;
        const int k = 2 * kp + sp2;
        const size_t set = (size_t)k * A.n_sel + si;
        const int gs = c * (po / n) + g;                   // subaperture within the item (column c * po + tid)
        const int q = it.q0 + gs, p = it.p + h;
        const bool inb = tid < po && gs < it.cnt && p < A.n_sub && k < A.n_steps;
        const int sa = inb ? p * A.n_sub + q : 0;
        const bool active = inb && A.valid[sa] != 0;
        if (!__any_sync(0xffffffffu, active)) continue;
        float binacc[2][P];                                // the two detector-row groups of this thread, before the exchange
#pragma unroll
        for (int hh = 0; hh < 2; ++hh)
#pragma unroll
            for (int i = 0; i < P; ++i) binacc[hh][i] = 0.0f;
        const float* ap = A.amp + (size_t)(p * n) * N + (size_t)q * n + b;
        uint32_t pht[ELONG ? n : 1];                       // ELONG: phase of the thread's column in 0.32 fixed-point turns
        if (ELONG) {
#pragma unroll
            for (int i = 0; i < n; ++i) {
                u64 v = acc[i];
#pragma unroll
                for (int hh = 1; hh < K::HS; ++hh) v = (hs == hh) ? acc[hh * n + i] : v;
                const float2 f = unpack2(v);
                float ph = (c ? f.y : f.x) * scale;
                if (MAPS && mp && active) ph += __ldg(mp + (size_t)(p * n + i) * N + (size_t)q * n + b);
                pht[ELONG ? i : 0] = phase_to_turns(ph);
            }
        }
        const int n_z = ELONG ? A.na.n_z : 1;
        const float* rho = ELONG ? A.na.rho + (size_t)((A.T.step0 + k) % A.na.n_t) * A.na.n_z : nullptr;
#pragma unroll 1
        for (int iz = 0; iz < n_z; ++iz) {
        __syncwarp();                                      // the previous round / scatterer has finished reading xs
        float wz = 1.0f;
        {
            float2 e[n];
            if (ELONG) {                                   // E = A exp(i (phi + ramp of scatterer iz)), reading O9
                const ElongRamp rp = elong_ramp(A.na, si, iz, p, q, n, N, sp.d);
                wz = __ldg(rho + iz);
                uint32_t t = (uint32_t)b * rp.fx;
#pragma unroll
                for (int i = 0; i < n; ++i) {
                    const float Am = active ? __ldg(ap + (size_t)i * N) : 0.0f;
                    float s, co;
                    sincos_turns(pht[ELONG ? i : 0] + t, &s, &co);
                    e[i] = make_float2(Am * co, Am * s);
                    t += rp.fy;
                }
            } else {
#pragma unroll
            for (int i = 0; i < n; ++i) {
                u64 v = acc[i];
#pragma unroll
                for (int hh = 1; hh < K::HS; ++hh) v = (hs == hh) ? acc[hh * n + i] : v;
                const float2 f = unpack2(v);
                float ph = (c ? f.y : f.x) * scale;
                if (MAPS && mp && active) ph += __ldg(mp + (size_t)(p * n + i) * N + (size_t)q * n + b);
                const float Am = active ? __ldg(ap + (size_t)i * N) : 0.0f;
                float s, co;
                sincos_reduced(ph, &s, &co);
                e[i] = make_float2(Am * co, Am * s);
            }
            }
            dft_half_padded<M>(e, [&](auto ki, const float2 v) {
                constexpr int kk = decltype(ki)::value;
                xs[kk * K::XP + b] = v;                    // column FFT result: T[k][b]
            });
        }
        __syncwarp();
        // rows k = b and k = b + n of this subaperture
#pragma unroll
        for (int hh = 0; hh < 2; ++hh) {
            const int kr = b + hh * n;
            float2 rrow[n];
#pragma unroll
            for (int i = 0; i < n; ++i) rrow[i] = xs[kr * K::XP + i];
            float bins[P];
#pragma unroll
            for (int i = 0; i < P; ++i) bins[i] = 0.0f;
            dft_half_padded<M>(rrow, [&](auto mi, const float2 v) {
                constexpr int m = decltype(mi)::value;
                bins[m / BETA] = fmaf(v.x, v.x, fmaf(v.y, v.y, bins[m / BETA]));
            });
#pragma unroll
            for (int i = 0; i < P; ++i) binacc[hh][i] = ELONG ? fmaf(wz, bins[i], binacc[hh][i]) : bins[i];
        }
        }
        float pixv[2][P];
        int cbase = 0;
#pragma unroll
        for (int hh = 0; hh < 2; ++hh) {
            float bins[P];
#pragma unroll
            for (int i = 0; i < P; ++i) bins[i] = binacc[hh][i];
            // sum the BETA rows of a detector row: halving exchange among BETA adjacent threads
            int cnt = P; cbase = 0;
#pragma unroll
            for (int mask = BETA / 2; mask >= 1; mask >>= 1) {
                const int half = cnt / 2;
                const bool up = (b & mask) != 0;
#pragma unroll
                for (int i = 0; i < P / 2; ++i) {
                    if (i < half) {
                        const float send = up ? bins[i] : bins[i + half];
                        const float keep = up ? bins[i + half] : bins[i];
                        bins[i] = keep + __shfl_xor_sync(0xffffffffu, send, mask);
                    }
                }
                if (up) cbase += half;
                cnt = half;
            }
#pragma unroll
            for (int i = 0; i < P; ++i) pixv[hh][i] = bins[i] * A.norm;
        }
        constexpr int NPIX = P / BETA;                     // pixels kept per row after the exchange
        // detector rows of this thread: r = (b + hh n) / BETA ; columns cbase .. cbase + NPIX - 1
        float s = 0.0f, mx = 0.0f, my = 0.0f;
        if (NOISE) {                                       // the thread's 2 NPIX pixels, long draws shared out over the warp
            float nv[2 * NPIX];
            uint32_t np[2 * NPIX];
#pragma unroll
            for (int hh = 0; hh < 2; ++hh)
#pragma unroll
                for (int i = 0; i < NPIX; ++i) {
                    nv[hh * NPIX + i] = pixv[hh][i];
                    np[hh * NPIX + i] = (uint32_t)(((b + hh * n) / BETA) * P + cbase + i);
                }
            __syncwarp();                                  // every lane has read its rows from xs: the warp's part is free
            noisy_pixels_warp<2 * NPIX>(nv, np, active, A.nz, (uint32_t)sa, (uint32_t)src_index, (uint32_t)(A.T.step0 + k),
                                        xch + (size_t)((tid & ~31) / n) * K::SUB_STRIDE);
#pragma unroll
            for (int hh = 0; hh < 2; ++hh)
#pragma unroll
                for (int i = 0; i < NPIX; ++i) pixv[hh][i] = nv[hh * NPIX + i];
        }
#pragma unroll
        for (int hh = 0; hh < 2; ++hh) {
            const int r = (b + hh * n) / BETA;
#pragma unroll
            for (int i = 0; i < NPIX; ++i) {
                float v = pixv[hh][i];
                const int col = cbase + i;
                if (A.images && active) A.images[(set * nsa + sa) * (P * P) + r * P + col] = v;
                s += v;
                mx = fmaf((float)col - 0.5f * (P - 1), v, mx);
                my = fmaf((float)r - 0.5f * (P - 1), v, my);
            }
        }
#pragma unroll
        for (int o = n / 2; o >= 1; o >>= 1) {
            s += __shfl_xor_sync(0xffffffffu, s, o);
            mx += __shfl_xor_sync(0xffffffffu, mx, o);
            my += __shfl_xor_sync(0xffffffffu, my, o);
        }
        if (A.slopes && active && b == 0) {
            const bool ok = fabsf(s) >= 1e-12f;
            A.slopes[(set * 2 + 0) * nsa + sa] = ok ? mx / s : 0.0f;
            A.slopes[(set * 2 + 1) * nsa + sa] = ok ? my / s : 0.0f;
        }
    }
}

// ------------------------------------------------------------------------------------------------
// k_fused64: the same fusion for M = 64 (n = 32 samples per subaperture, 8 x 8 pixels of 8 x 8 FFT pixels; c4's largest
// sweep point).  A work item is one subaperture row of up to 8 adjacent subapertures = 32 x 256 samples, for two steps.
// The 16-row tile of trace2.cuh is marched twice: the top half's sums go to a shared-memory stash (each thread reads
// back only what it wrote), the bottom half stays in registers.  The two halves carry different warp-uniform piston
// references; their FP64 difference is added to the top half so that a subaperture has ONE piston (which |FFT|^2 does
// not see).  Image formation: one warp per subaperture and round (step, column half): thread b holds column b
// (32 samples), two 32-point FFTs in registers (dft_half_padded<64>), transpose through shared memory, rows b and
// b + 32, |.|^2, 8 x 8 binning (8 columns in registers, 8 rows through shared memory), noise, centre of gravity.
constexpr int kF64Stash = kKS * kTR * kTileCols * (int)sizeof(float);                 // 32 KB
constexpr int kF64XP = 33;                                                              // transpose pitch, float2
constexpr int kF64Sub = 64 * kF64XP * (int)sizeof(float2) + (64 * 8 + 64) * (int)sizeof(float);   // per warp: T[64][33], row bins, pixels
constexpr size_t kF64Xch = 4 * (size_t)kF64Sub;

template <int MODE, bool NOISE>
__global__ void __launch_bounds__(kFusedThreads, 2)
k_fused64(const FusedArgs A, const unsigned stash_off)
{
    constexpr int M = 64, n = 32, P = 8, BETA = 8, NT = kFusedThreads;
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ Trace2Shared S;
    const int tid = threadIdx.x, warp = tid >> 5, b = tid & 31;
    const int kp = (int)(blockIdx.x % (unsigned)A.n_pairs);
    const unsigned rest = blockIdx.x / (unsigned)A.n_pairs;
    const WorkItem it = A.items[rest % (unsigned)A.n_items];
    const int si = (int)(rest / (unsigned)A.n_items);
    const int src_index = A.sel[si];
    const SourceP sp = A.T.srcs[src_index];
    const int N = A.n_sub * n, nsa = A.n_sub * A.n_sub;
    float* stash = reinterpret_cast<float*>(smem + stash_off);     // [step][row < 16][column < 256]

    u64 acc[kKS * kTR];
    double rs_top[2] = {0.0, 0.0}, rs_bot[2] = {0.0, 0.0};
#pragma unroll 1
    for (int half = 0; half < 2; ++half) {                 // one copy of the march in the code: the kernel is 180 KB of SASS as it is
        double rs[2];
        trace2_tile<NT, true, MODE>(A.T, sp, S, smem, it.q0 * n, it.p * n + half * kTR, A.T.step0 + 2 * kp, acc, rs);
        if (half == 0) {
            rs_top[0] = rs[0]; rs_top[1] = rs[1];
#pragma unroll
            for (int i = 0; i < kKS * kTR; ++i) {
                const float2 f = unpack2(acc[i]);
                stash[i * kTileCols + tid] = f.x;
                stash[i * kTileCols + NT + tid] = f.y;
            }
        } else { rs_bot[0] = rs[0]; rs_bot[1] = rs[1]; }
        __syncthreads();                                   // every warp has left the march: barriers and stages are re-armed / dead
    }
    const float dref[2] = {(float)(rs_top[0] - rs_bot[0]), (float)(rs_top[1] - rs_bot[1])};

    unsigned char* wbuf = smem + (size_t)warp * kF64Sub;
    float2* xs = reinterpret_cast<float2*>(wbuf);                              // T[k][b]
    float* rb = reinterpret_cast<float*>(wbuf + 64 * kF64XP * sizeof(float2));   // row bins [64][8]
    float* pix = rb + 64 * 8;
    const float scale = (float)sp.scale;
    const float* mp = sp.map;
    const int p = it.p;
#pragma unroll 1
    for (int rd = 0; rd < 4; ++rd) {
        const int s2 = rd >> 1, c = rd & 1;                // step in pair, column half: subaperture c * 4 + warp of the item
        const int k = 2 * kp + s2;
        const size_t set = (size_t)k * A.n_sel + si;
        const int gs = c * 4 + warp, q = it.q0 + gs;
        const bool inb = gs < it.cnt && k < A.n_steps;
        const int sa = inb ? p * A.n_sub + q : 0;
        const bool active = inb && A.valid[sa] != 0;      // warp-uniform
        if (!active) continue;
        __syncwarp();                                      // the previous round has finished reading xs
        {
            float2 e[n];
            const float* ap = A.amp + (size_t)(p * n) * N + (size_t)q * n + b;
            const float* st = stash + (size_t)(s2 * kTR) * kTileCols + c * NT + tid;
#pragma unroll
            for (int i = 0; i < n; ++i) {
                float ph;
                if (i < kTR) ph = st[i * kTileCols] + dref[c];
                else {
                    const float2 f = unpack2(s2 ? acc[kTR + i - kTR] : acc[i - kTR]);
                    ph = c ? f.y : f.x;
                }
                ph *= scale;
                if (mp) ph += __ldg(mp + (size_t)(p * n + i) * N + (size_t)q * n + b);
                const float Am = __ldg(ap + (size_t)i * N);
                float sn, co;
                sincos_reduced(ph, &sn, &co);
                e[i] = make_float2(Am * co, Am * sn);
            }
            dft_half_padded<M>(e, [&](auto ki, const float2 v) {
                constexpr int kk = decltype(ki)::value;
                xs[kk * kF64XP + b] = v;
            });
        }
        __syncwarp();
#pragma unroll
        for (int hh = 0; hh < 2; ++hh) {                   // rows b and b + 32
            const int kr = b + hh * n;
            float2 rrow[n];
#pragma unroll
            for (int i = 0; i < n; ++i) rrow[i] = xs[kr * kF64XP + i];
            float bins[P];
#pragma unroll
            for (int i = 0; i < P; ++i) bins[i] = 0.0f;
            dft_half_padded<M>(rrow, [&](auto mi, const float2 v) {
                constexpr int m = decltype(mi)::value;
                bins[m / BETA] = fmaf(v.x, v.x, fmaf(v.y, v.y, bins[m / BETA]));
            });
#pragma unroll
            for (int i = 0; i < P; ++i) rb[kr * P + i] = bins[i];
        }
        __syncwarp();
        float s = 0.0f, mx = 0.0f, my = 0.0f;
#pragma unroll
        for (int t = 0; t < 2; ++t) {                      // pixels b and b + 32: sum of their 8 rows
            const int px = b + t * 32, r = px >> 3, col = px & 7;
            float v = 0.0f;
#pragma unroll
            for (int y = 0; y < BETA; ++y) v += rb[(r * BETA + y) * P + col];
            v *= A.norm;
            if (NOISE) v = noisy_pixel(v, A.nz, (uint32_t)px, (uint32_t)sa, (uint32_t)src_index, (uint32_t)(A.T.step0 + k));
            if (A.images) A.images[(set * nsa + sa) * (P * P) + px] = v;
            s += v;
            mx = fmaf((float)col - 0.5f * (P - 1), v, mx);
            my = fmaf((float)r - 0.5f * (P - 1), v, my);
        }
#pragma unroll
        for (int o = 16; o >= 1; o >>= 1) {
            s += __shfl_xor_sync(0xffffffffu, s, o);
            mx += __shfl_xor_sync(0xffffffffu, mx, o);
            my += __shfl_xor_sync(0xffffffffu, my, o);
        }
        if (A.slopes && b == 0) {
            const bool ok = fabsf(s) >= 1e-12f;
            A.slopes[(set * 2 + 0) * nsa + sa] = ok ? mx / s : 0.0f;
            A.slopes[(set * 2 + 1) * nsa + sa] = ok ? my / s : 0.0f;
        }
    }
}

// ------------------------------------------------------------------------------------------------
// host side
// Tile shape of the fused kernel per FFT size: G subapertures wide, R2 subaperture rows tall.
void fused_tile_shape(int M, int* G, int* R2)
{
    if (M == 32) { *G = FusedCfg<32>::G; *R2 = FusedCfg<32>::R2; }
    else if (M == 16) { *G = FusedCfg<16>::G; *R2 = FusedCfg<16>::R2; }
    else if (M == 64) { *G = kTileCols / 32; *R2 = 1; }            // k_fused64: one subaperture row of 8 per work item
    else { *G = 0; *R2 = 0; }
}

static size_t fused_xch_bytes(int M) { return M == 64 ? kF64Xch : M == 32 ? FusedCfg<32>::XCH_BYTES : FusedCfg<16>::XCH_BYTES; }
#ifndef AO_FUSED_BUDGET_KB
#define AO_FUSED_BUDGET_KB 72
#endif
// shared-memory budget per CTA: three CTAs per SM (168 registers, no spills: measured 141 us against 148 at four CTAs of 128
// registers and 155 at two CTAs of 204 on c4 / M = 32), M = 64 two CTAs per SM
static size_t fused_budget(int M) { return M == 64 ? 72 * 1024 : (size_t)AO_FUSED_BUDGET_KB * 1024; }

// cuTensorMapEncodeTiled through the runtime's driver entry point (no link against libcuda); NULL if unavailable.
static PFN_cuTensorMapEncodeTiled tensor_map_encoder()
{
    static PFN_cuTensorMapEncodeTiled fn = []() -> PFN_cuTensorMapEncodeTiled {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess ||
            q != cudaDriverEntryPointSuccess) { cudaGetLastError(); return nullptr; }
        return (PFN_cuTensorMapEncodeTiled)p;
    }();
    return fn;
}

// One tensor map per layer over the borrowed screen [S][S], each with its OWN box {pitch_l, rows_l} (the extent of a tile
// on that layer: du and the wind shift differ per layer, so a common box would overfetch): the staged box of a tile is
// then a single cp.async.bulk.tensor.2d (UTMALDG) instead of one bulk copy per row.  Encoded once per (plan, dt), cached.
static cudaError_t ensure_tensor_maps(ao_geometry* g, WfsH& w, const Tile2Plan& pl, double dt, cudaStream_t st)
{
    if (w.tm_pitch == pl.pitch && w.tm_rows == pl.rows && w.tm_dt == dt) return cudaSuccess;
    PFN_cuTensorMapEncodeTiled enc = tensor_map_encoder();
    if (!enc || !w.d_tmaps) return cudaErrorNotSupported;
    const size_t nl = g->layers.size();
    std::vector<unsigned char> buf(nl * (sizeof(CUtensorMap) + sizeof(int2)));
    CUtensorMap* maps = reinterpret_cast<CUtensorMap*>(buf.data());
    int2* boxes = reinterpret_cast<int2*>(buf.data() + nl * sizeof(CUtensorMap));
    for (size_t l = 0; l < nl; ++l) {
        const LayerP& lp = g->layers[l];
        // this layer's own box: the extent of a tile over the two paired steps, as in plan_tiles2 but per layer
        double ext_x = 0.0, ext_y = 0.0;
        for (int s : w.grp.src) {
            const SourceP& sp = g->sources[s];
            if (!(lp.height < sp.H)) continue;
            double du = (1.0 - lp.height * sp.inv_H) * sp.d * lp.inv_pitch;
            if (fabs(du - 1.0) < 1e-9) du = 1.0;
            ext_x = std::max(ext_x, (kTileCols - 1) * du + fabs(lp.wx * dt * lp.inv_pitch) * (kKS - 1));
            ext_y = std::max(ext_y, (kTR - 1) * du + fabs(lp.wy * dt * lp.inv_pitch) * (kKS - 1));
        }
        int pt = std::min(pl.pitch, (((int)ceil(ext_x) + 8) + 7) & ~7);
        int rw = std::min(pl.rows, (int)ceil(ext_y) + 3 + (pl.quad ? 2 : 0));
        if (pt < 8) pt = 8;
        if (rw < 1) rw = 1;
        boxes[l] = make_int2(pt, rw);
        const cuuint64_t dims[2] = {(cuuint64_t)lp.S, (cuuint64_t)lp.S};
        const cuuint64_t strides[1] = {(cuuint64_t)lp.S * sizeof(float)};
        const cuuint32_t box[2] = {(cuuint32_t)pt, (cuuint32_t)rw};
        const cuuint32_t estr[2] = {1, 1};
        if (lp.S < pt || lp.S < rw ||
            enc(&maps[l], CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, (void*)lp.screen, dims, strides, box, estr,
                CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
            return cudaErrorNotSupported;
    }
    static_assert(sizeof(CUtensorMap) == 128, "tensor maps are indexed by 128 bytes in trace2.cuh");
    cudaError_t e = cudaMemcpyAsync(w.d_tmaps, buf.data(), buf.size(), cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) { w.tm_pitch = pl.pitch; w.tm_rows = pl.rows; w.tm_dt = dt; }
    return e;
}

bool fused_supported(const ao_geometry* g, const WfsH& w, double dt)
{
    if (!(w.M == 16 || w.M == 32 || w.M == 64) || w.n * 2 != w.M || w.P != 8 || w.beta * w.P != w.M) return false;
    if (w.fused_items == nullptr || w.n_fused_items == 0) return false;
    if (w.M == 64 && w.na.n_z > 0) return false;           // extended beacons at M = 64 run k_sh_generic
    const Tile2Plan pl = plan_tiles2(g, w.grp.src, dt, fused_xch_bytes(w.M), fused_budget(w.M));
    return pl.ok && (w.M != 64 || pl.smem + 128 + kF64Stash <= 113 * 1024);
}

template <int M>
static cudaError_t launch_fused_variant(ao_geometry* g, const WfsH& w, FusedArgs a, const Tile2Plan& pl, int n_steps,
                                        cudaStream_t st)
{
    bool maps = false;                                     // the map-free kernel keeps its register budget
    for (int si : w.grp.src) maps = maps || g->sources[si].map != nullptr;
    void (*kern)(const FusedArgs);
    if (a.na.n_z > 0)       // extended beacon: its own instantiations (they also read the phase maps if any are set)
        kern = pl.anydu ? (a.nz.on ? k_fused<M, true, true, true, true> : k_fused<M, false, true, true, true>)
                        : (a.nz.on ? k_fused<M, true, false, true, true> : k_fused<M, false, false, true, true>);
    else if (maps) kern = pl.anydu ? (a.nz.on ? k_fused<M, true, true, true, false> : k_fused<M, false, true, true, false>)
                                   : (a.nz.on ? k_fused<M, true, false, true, false> : k_fused<M, false, false, true, false>);
    else kern = pl.anydu ? (a.nz.on ? k_fused<M, true, true, false, false> : k_fused<M, false, true, false, false>)
                         : (a.nz.on ? k_fused<M, true, false, false, false> : k_fused<M, false, false, false, false>);
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl.smem);
    if (e != cudaSuccess) return e;
    const size_t nsa = (size_t)w.n_sub * w.n_sub;
    const long long per_pair = (long long)a.n_items * a.n_sel;
    int max_steps = (int)std::max<long long>(2, 2 * (0x7fffffffLL / per_pair));
    max_steps &= ~1;                                       // chunks start on an even step: pairs stay aligned
    const int64_t step0 = a.T.step0;
    for (int k0 = 0; k0 < n_steps; k0 += max_steps) {
        const int ks = n_steps - k0 < max_steps ? n_steps - k0 : max_steps;
        FusedArgs b = a;
        b.T.step0 = step0 + k0; b.n_steps = ks; b.n_pairs = (ks + kKS - 1) / kKS;
        const size_t set0 = (size_t)k0 * a.n_sel;
        if (a.images) b.images = a.images + set0 * nsa * w.P * w.P;
        if (a.slopes) b.slopes = a.slopes + set0 * 2 * nsa;
        kern<<<(unsigned)(per_pair * b.n_pairs), kFusedThreads, pl.smem, st>>>(b);
        g->launches++;
        if ((e = cudaGetLastError()) != cudaSuccess) return e;
    }
    return cudaSuccess;
}

static cudaError_t launch_fused64(ao_geometry* g, const WfsH& w, FusedArgs a, const Tile2Plan& pl, int n_steps, cudaStream_t st)
{
    void (*kern)(const FusedArgs, const unsigned);
    const int mode = pl.quad ? 2 : (pl.anydu ? 1 : 0);
    if (a.nz.on) kern = mode == 2 ? k_fused64<2, true> : mode == 1 ? k_fused64<1, true> : k_fused64<0, true>;
    else kern = mode == 2 ? k_fused64<2, false> : mode == 1 ? k_fused64<1, false> : k_fused64<0, false>;
    const unsigned stash_off = (unsigned)((pl.smem + 127) & ~(size_t)127);
    const size_t smem = (size_t)stash_off + kF64Stash;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const size_t nsa = (size_t)w.n_sub * w.n_sub;
    const long long per_pair = (long long)a.n_items * a.n_sel;
    int max_steps = (int)std::max<long long>(2, 2 * (0x7fffffffLL / per_pair));
    max_steps &= ~1;
    const int64_t step0 = a.T.step0;
    for (int k0 = 0; k0 < n_steps; k0 += max_steps) {
        const int ks = n_steps - k0 < max_steps ? n_steps - k0 : max_steps;
        FusedArgs b = a;
        b.T.step0 = step0 + k0; b.n_steps = ks; b.n_pairs = (ks + kKS - 1) / kKS;
        const size_t set0 = (size_t)k0 * a.n_sel;
        if (a.images) b.images = a.images + set0 * nsa * w.P * w.P;
        if (a.slopes) b.slopes = a.slopes + set0 * 2 * nsa;
        kern<<<(unsigned)(per_pair * b.n_pairs), kFusedThreads, smem, st>>>(b, stash_off);
        g->launches++;
        if ((e = cudaGetLastError()) != cudaSuccess) return e;
    }
    return cudaSuccess;
}

cudaError_t launch_fused(ao_geometry* g, const WfsH& w, int64_t step0, int n_steps, double dt,
                         const NoiseP& noise, float* images, float* slopes, cudaStream_t st)
{
    if (!fused_supported(g, w, dt)) return cudaErrorNotSupported;
    Tile2Plan pl = plan_tiles2(g, w.grp.src, dt, fused_xch_bytes(w.M), fused_budget(w.M), w.d_tmaps != nullptr);
    if (pl.tma && (!pl.ok || ensure_tensor_maps(g, const_cast<WfsH&>(w), pl, dt, st) != cudaSuccess)) {
        cudaGetLastError();
        pl = plan_tiles2(g, w.grp.src, dt, fused_xch_bytes(w.M), fused_budget(w.M));      // per-row bulk copies
    }
    const size_t n_sel = w.grp.src.size(), nsa = (size_t)w.n_sub * w.n_sub;
    cudaError_t e;
    // invalid subapertures are never scheduled: zero-fill the outputs first
    if (images && (e = cudaMemsetAsync(images, 0, sizeof(float) * n_steps * n_sel * nsa * w.P * w.P, st)) != cudaSuccess) return e;
    if (slopes && (e = cudaMemsetAsync(slopes, 0, sizeof(float) * n_steps * n_sel * 2 * nsa, st)) != cudaSuccess) return e;
    FusedArgs a;
    a.T = make_trace2_args(g, pl, step0, dt);
    if (pl.tma) a.T.tmaps = w.d_tmaps;
    a.sel = w.grp.d_src; a.n_sel = (int)n_sel;
    a.items = (const WorkItem*)w.fused_items; a.n_items = w.n_fused_items; a.n_steps = n_steps;
    a.amp = w.d_amp; a.valid = w.d_valid; a.n_sub = w.n_sub;
    a.norm = (float)(1.0 / ((double)w.M * w.M * (double)w.n * w.n));
    a.nz = noise; a.images = images; a.slopes = slopes; a.na = w.na;
    if (w.M == 64) return launch_fused64(g, w, a, pl, n_steps, st);
    if (w.M == 32) return launch_fused_variant<32>(g, w, a, pl, n_steps, st);
    return launch_fused_variant<16>(g, w, a, pl, n_steps, st);
}

}  // namespace ao
