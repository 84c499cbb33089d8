// k_fused.cu -- the WFS hot path: ray-trace + Shack-Hartmann image + centre of gravity in ONE kernel
// (ao_sh_images with phase_dev == NULL for M in {16, 32}, n = M/2, beta*P = M; PAPER.md:56,60,28,82;
// readings O2, O3, O4, O5, O6).  Phase never touches HBM.
//
// Work decomposition.  A CTA processes one work item = a run of up to G horizontally adjacent VALID
// subapertures of one (step, source): an n-row x (G n)-column tile of phase samples.  Invalid
// subapertures are never scheduled (their outputs are zero-filled by a memset).
//
// Phase A, ray-trace (per layer):  the screen footprint of the tile ((n-1) dv + 3 rows by
// (G n - 1) du + 6 columns) is staged in shared memory by the TMA engine: the lanes of warp 0 issue one
// cp.async.bulk row copy each (periodic wrap handled per row / per segment), completing on an mbarrier;
// NS stages are in flight so the copies of layer l+NS-1 overlap the arithmetic of layer l.
// Each thread owns C columns of the tile and marches down the n rows: the bilinear interpolation is
// separable, so the x-interpolated screen rows X_r = s[r][j0] + fx (s[r][j0+1] - s[r][j0]) are computed once
// per screen row (du, dv <= 1: fewer screen rows than output rows) and the y-interpolation
// acc_i += (1-fy) X_r + fy X_{r+1} costs two FFMAs per sample.  Precision: the column coordinate is
// FP64 per (thread, layer); the row coordinate advances in fp32 from an FP64 origin (|error| < 1e-6 px
// over n <= 32 rows); a per-(subaperture, layer) piston reference is subtracted from every tap so that
// all fp32 sums stay at the few-radian level (|E~|^2 is piston-invariant).
//
// Phase B, image formation (per slot of G/C subapertures):  thread (g, b) holds column b of subaperture
// g: E[a] = A exp(i phi).  Column FFTs run entirely in registers: the half-pixel-centred, zero-padded
// M-point DFT of n inputs splits (first DIF stage on half-zero input) into two n-point FFTs of
// e[a] cis(pi (M-1) a/M) and e[a] cis(pi (M-3) a/M) with compile-time twiddles.  One transpose through
// padded shared memory, then the row FFTs (two rows per thread), |.|^2, beta x beta binning (in-register
// over m, halving shuffles over k), optional noise, centre of gravity by warp shuffles.
#include <type_traits>

#include "ao_device.cuh"

namespace ao {

// ------------------------------------------------------------------------------------------------
// compile-time trigonometry and complex constants
constexpr double kPi = 3.14159265358979323846264338327950288;
constexpr double cx_sin(double x)
{
    double t = x, s = x;
    for (int i = 1; i < 28; ++i) { t *= -x * x / ((2.0 * i) * (2.0 * i + 1.0)); s += t; }
    return s;
}
constexpr double cx_cos(double x)
{
    double t = 1.0, s = 1.0;
    for (int i = 1; i < 28; ++i) { t *= -x * x / ((2.0 * i - 1.0) * (2.0 * i)); s += t; }
    return s;
}

// cis(pi NUM / DEN) as compile-time floats
template <int NUM, int DEN>
struct Cis {
    static constexpr int q = ((NUM % (2 * DEN)) + 2 * DEN) % (2 * DEN);       // angle = pi q / DEN in [0, 2 pi)
    static constexpr int qs = q >= DEN ? q - 2 * DEN : q;                      // in [-pi, pi)
    static constexpr float re = (float)cx_cos(kPi * (double)qs / (double)DEN);
    static constexpr float im = (float)cx_sin(kPi * (double)qs / (double)DEN);
};

template <int NUM, int DEN>
__device__ __forceinline__ float2 cmul_cis(const float2 x)
{
    using W = Cis<NUM, DEN>;
    if constexpr (W::q == 0) return x;
    else if constexpr (2 * W::q == DEN) return make_float2(-x.y, x.x);
    else if constexpr (W::q == DEN) return make_float2(-x.x, -x.y);
    else if constexpr (2 * W::q == 3 * DEN) return make_float2(x.y, -x.x);
    else return make_float2(fmaf(x.x, W::re, -x.y * W::im), fmaf(x.x, W::im, x.y * W::re));
}

template <int I, int N, typename F>
__device__ __forceinline__ void static_for(F&& f)
{
    if constexpr (I < N) {
        f(std::integral_constant<int, I>{});
        static_for<I + 1, N>(static_cast<F&&>(f));
    }
}

__host__ __device__ constexpr int bitrev_c(int k, int n)
{
    int r = 0;
    for (int b = 1; b < n; b <<= 1) { r = (r << 1) | (k & 1); k >>= 1; }
    return r;
}

// In-register radix-2 DIF FFT, forward sign, natural-order input, X[k] = x[bitrev(k)] on output.
template <int N, int HALF>
__device__ __forceinline__ void fft_stage(float2 (&x)[N])
{
    static_for<0, N / 2>([&](auto bi) {
        constexpr int b = decltype(bi)::value;
        constexpr int grp = b / HALF, pos = b % HALF, i = grp * 2 * HALF + pos, j = i + HALF;
        const float2 a = x[i], c = x[j];
        x[i] = make_float2(a.x + c.x, a.y + c.y);
        x[j] = cmul_cis<-pos, HALF>(make_float2(a.x - c.x, a.y - c.y));      // * exp(-2 pi i pos/(2 HALF))
    });
    if constexpr (HALF > 1) fft_stage<N, HALF / 2>(x);
}

// Half-pixel-centred DFT of size M = 2n of n inputs (zero padded):
//   X[k] = sum_a e[a] exp(-2 pi i (k - (M-1)/2) a / M),  k < M.
// First DIF stage on the half-zero input: X[2k'] = FFT_n(e[a] cis(pi (M-1) a/M))[k'],
//                                         X[2k'+1] = FFT_n(e[a] cis(pi (M-3) a/M))[k'].
// `sink(k, value)` is called once for every k (k as std::integral_constant).
template <int M, typename Sink>
__device__ __forceinline__ void dft_half_padded(const float2 (&e)[M / 2], Sink&& sink)
{
    constexpr int n = M / 2;
    float2 y[n];
    static_for<0, n>([&](auto ai) { constexpr int a = decltype(ai)::value; y[a] = cmul_cis<(M - 1) * a, M>(e[a]); });
    fft_stage<n, n / 2>(y);
    static_for<0, n>([&](auto ki) { constexpr int k = decltype(ki)::value; sink(std::integral_constant<int, 2 * k>{}, y[bitrev_c(k, n)]); });
    static_for<0, n>([&](auto ai) { constexpr int a = decltype(ai)::value; y[a] = cmul_cis<(M - 3) * a, M>(e[a]); });
    fft_stage<n, n / 2>(y);
    static_for<0, n>([&](auto ki) { constexpr int k = decltype(ki)::value; sink(std::integral_constant<int, 2 * k + 1>{}, y[bitrev_c(k, n)]); });
}

// ------------------------------------------------------------------------------------------------
// mbarrier / TMA bulk-copy PTX
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

struct WorkItem { int p, q0, cnt, pad; };

struct FusedArgs {
    const LayerP* layers; int n_layers;
    const SourceP* srcs; const int* sel; int n_sel;
    const WorkItem* items;
    const float* amp;                 // [N][N] on the WFS grid
    const uint8_t* valid;             // [n_sub^2]
    int n_sub;
    long long step0; double dt;
    float norm;                       // 1/(M^2 n^2)
    NoiseP nz;
    float* images;                    // nullable [k][si][nsa][P][P]
    float* slopes;                    // nullable [k][si][2][nsa]
};

// M: FFT size (n = M/2 samples per subaperture side); G: subapertures per tile row; C: columns per
// thread; R2: subaperture rows per tile.
template <int M, int G, int C, int R2>
struct FusedCfg {
    static constexpr int n = M / 2;
    static constexpr int NR = R2 * n;                    // tile rows (<= 32: one lane per row)
    static constexpr int NCOL = G * n;                   // tile columns
    static constexpr int NT = NCOL / C;                  // threads per CTA
    static constexpr int GS = NT / n;                    // subapertures per FFT round
    static constexpr int P = 8, BETA = M / 8;
    static constexpr int PITCH = NCOL + 8;               // staged tile row pitch in floats (du <= 1)
    static constexpr int RMAX = NR + 2;                  // staged tile rows (dv <= 1)
    static constexpr int XP = n + 1;                     // transpose pitch (float2 units)
    static constexpr int SUB_STRIDE = M * XP + (n == 8 ? 8 : 0);
    static constexpr int NS = 3;                         // TMA stages
    static constexpr size_t TILE_BYTES = (size_t)NS * RMAX * PITCH * sizeof(float);
    static constexpr size_t XCH_BYTES = (size_t)GS * SUB_STRIDE * sizeof(float2);
    static constexpr size_t SMEM = (TILE_BYTES > XCH_BYTES ? TILE_BYTES : XCH_BYTES) + 128;
    static_assert(NR <= 32 && NCOL % C == 0 && NT % 32 == 0, "bad fused configuration");
};

template <int M, int G, int C, int R2, bool NOISE>
__global__ void __launch_bounds__(FusedCfg<M, G, C, R2>::NT)
k_fused(const FusedArgs A)
{
    using K = FusedCfg<M, G, C, R2>;
    constexpr int n = K::n, NR = K::NR, NT = K::NT, NS = K::NS, P = K::P, BETA = K::BETA, PITCH = K::PITCH;
    constexpr int TILE_FLOATS = K::RMAX * PITCH;
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ uint64_t full_bar[NS];
    __shared__ double s_u0[kMaxLayers], s_du[kMaxLayers], s_v0[kMaxLayers], s_c0[kMaxLayers];
    __shared__ int s_wt[kMaxLayers], s_rt[kMaxLayers], s_act[kMaxLayers], s_nact;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const WorkItem it = A.items[blockIdx.x];
    const int si = blockIdx.y, k = blockIdx.z;
    const int src_index = A.sel[si];
    const SourceP sp = A.srcs[src_index];
    const int N = A.n_sub * n, nsa = A.n_sub * A.n_sub;
    float* tiles = reinterpret_cast<float*>(smem);                     // [NS][RMAX][PITCH]
    float2* xch = reinterpret_cast<float2*>(smem);                     // reused after the trace
    const int jfirst = it.q0 * n, ifirst = it.p * n;                   // tile origin on the WFS grid

    // ---- per-CTA layer table (FP64): column origin/increment, row origin, staged box ----
    if (tid == 0) {
        int na = 0;
        for (int l = 0; l < A.n_layers; ++l)
            if (A.layers[l].height < sp.H) s_act[na++] = l;
        s_nact = na;
#pragma unroll
        for (int s = 0; s < NS; ++s) mbar_init(&full_bar[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    {
        const double t = (double)(A.step0 + k) * A.dt;
        for (int l = tid; l < A.n_layers; l += NT) {
            const LayerP lp = A.layers[l];
            const double gamma = 1.0 - lp.height * sp.inv_H;
            const double x0 = -0.5 * (double)(sp.N - 1) * sp.d;
            const double c = 0.5 * (double)(lp.S - 1);
            const double du = gamma * sp.d * lp.inv_pitch;
            const double u0 = (gamma * x0 + lp.height * sp.thx - lp.wx * t) * lp.inv_pitch + c;
            const double v0 = (gamma * x0 + lp.height * sp.thy - lp.wy * t) * lp.inv_pitch + c;
            const double vrow0 = fma((double)ifirst, du, v0);                       // row coordinate of tile row 0
            const long long c0 = (long long)floor(fma((double)jfirst, du, u0)) & ~3LL;   // 16-byte aligned start
            const long long clast = (long long)floor(fma((double)(jfirst + K::NCOL - 1), du, u0)) + 2;
            const long long rlast = (long long)floor(fma((double)(ifirst + NR - 1), du, v0)) + 2;
            int wt = (int)(clast - c0 + 1); wt = (wt + 3) & ~3; if (wt > PITCH) wt = PITCH;
            int rt = (int)(rlast - (long long)floor(vrow0) + 1); if (rt > K::RMAX) rt = K::RMAX;
            s_u0[l] = u0; s_du[l] = du; s_v0[l] = vrow0; s_c0[l] = (double)c0; s_wt[l] = wt; s_rt[l] = rt;
        }
    }
    __syncthreads();
    const int nact = s_nact;

    // producer: the lanes of warp 0 copy the rows of layer ordinal `a` into stage a % NS (TMA bulk copies)
    auto issue = [&](int a) {
        const int l = s_act[a];
        const LayerP lp = A.layers[l];
        const int wt = s_wt[l], rt = s_rt[l];
        const long long c0 = (long long)s_c0[l];
        const long long r0 = (long long)floor(s_v0[l]);
        uint64_t* bar = &full_bar[a % NS];
        float* dst = tiles + (size_t)(a % NS) * TILE_FLOATS;
        if (lane == 0) mbar_expect_tx(bar, (uint32_t)(rt * wt) * 4u);
        __syncwarp();
        long long cw = c0 % lp.S; if (cw < 0) cw += lp.S;
        const int first = (cw + wt <= lp.S) ? wt : (int)(lp.S - cw);          // floats before the periodic wrap
        for (int r = lane; r < rt; r += 32) {
            long long rr = (r0 + r) % lp.S; if (rr < 0) rr += lp.S;
            const float* srow = lp.screen + (size_t)rr * lp.S;
            bulk_g2s(dst + r * PITCH, srow + cw, (uint32_t)first * 4u, bar);
            if (first < wt) bulk_g2s(dst + r * PITCH + first, srow, (uint32_t)(wt - first) * 4u, bar);
        }
    };
    if (warp == 0)
        for (int a = 0; a < NS && a < nact; ++a) issue(a);

    // ---- phase A: ray-trace into registers ----
    float acc[C][NR];
#pragma unroll
    for (int c = 0; c < C; ++c)
#pragma unroll
        for (int i = 0; i < NR; ++i) acc[c][i] = 0.0f;

    // Per-layer coordinates, computed one layer ahead of use (FP64, off the critical path):
    //   rowcode: lane i holds fy_i of tile row i, sign bit set iff the screen row advances before row i
    //   jrel/fx: cell (relative to the staged box) and fraction of each of this thread's columns
    struct LayerCoord { float rowcode; int jrel[C]; float fx[C]; };
    auto coords = [&](int a) {
        LayerCoord lc;
        const int l = s_act[a];
        const double du = s_du[l], u0 = s_u0[l], c0d = s_c0[l], vrow0 = s_v0[l];
        {
            const double v = fma((double)lane, du, vrow0);
            const double vfl = floor(v);
            float fy = (float)(v - vfl);
            int r = (int)(vfl - floor(vrow0));
            if (fy >= 1.0f) { fy = 0.0f; ++r; }
            const int rprev = __shfl_up_sync(0xffffffffu, r, 1);
            const bool adv = lane > 0 && r != rprev;
            lc.rowcode = adv ? -fy : fy;                 // -0.0f keeps the sign bit when fy == 0
        }
#pragma unroll
        for (int c = 0; c < C; ++c) {
            const double u = fma((double)(jfirst + c * NT + tid), du, u0);
            const double uf = floor(u);
            lc.fx[c] = (float)(u - uf);
            lc.jrel[c] = (int)(uf - c0d);
            if (lc.fx[c] >= 1.0f) { lc.fx[c] = 0.0f; ++lc.jrel[c]; }
        }
        return lc;
    };
    LayerCoord cur = {};
    if (nact > 0) cur = coords(0);
    const uint32_t tiles_s = smem_u32(tiles);
    constexpr uint32_t PB = PITCH * 4;                     // staged row pitch in bytes

    for (int a = 0; a < nact; ++a) {
        LayerCoord nxt = cur;
        if (a + 1 < nact) nxt = coords(a + 1);
        const uint32_t tile_s = tiles_s + (uint32_t)(a % NS) * (uint32_t)(TILE_FLOATS * 4);
        const float* tile = tiles + (size_t)(a % NS) * TILE_FLOATS;
        mbar_wait(&full_bar[a % NS], (uint32_t)((a / NS) & 1));
        uint32_t tp[C]; float T[C], B[C], ref[C];
#pragma unroll
        for (int c = 0; c < C; ++c) {
            // piston reference: first tap of the subaperture's first column (same for its n threads)
            const int jref = __shfl_sync(0xffffffffu, cur.jrel[c], lane & ~(n - 1) & 31);
            ref[c] = tile[jref];
            const float* t0 = tile + cur.jrel[c];
            const float s0 = t0[0], s1 = t0[1], s2 = t0[PITCH], s3 = t0[PITCH + 1];
            T[c] = fmaf(cur.fx[c], s1 - s0, s0 - ref[c]);
            B[c] = fmaf(cur.fx[c], s3 - s2, s2 - ref[c]);
            tp[c] = tile_s + (uint32_t)cur.jrel[c] * 4u;
        }
#pragma unroll
        for (int i = 0; i < NR; ++i) {
            const float code = __shfl_sync(0xffffffffu, cur.rowcode, i);     // warp-uniform
            if (i > 0) {
                // advance one screen row when the sign bit is set; bra.uni: the predicate is warp-uniform
                if constexpr (C == 1) {
                    asm volatile(
                        "{\n\t.reg .pred p;\n\t.reg .f32 s0, s1;\n\t"
                        "setp.lt.s32 p, %3, 0;\n\t"
                        "@!p bra.uni SKIP_%=;\n\t"
                        "add.u32 %0, %0, %6;\n\t"
                        "ld.shared.f32 s0, [%0+%6];\n\t"
                        "ld.shared.f32 s1, [%0+%7];\n\t"
                        "mov.f32 %1, %2;\n\t"
                        "sub.f32 s1, s1, s0;\n\t"
                        "sub.f32 s0, s0, %4;\n\t"
                        "fma.rn.f32 %2, %5, s1, s0;\n\t"
                        "SKIP_%=:\n\t}"
                        : "+r"(tp[0]), "+f"(T[0]), "+f"(B[0])
                        : "r"(__float_as_int(code)), "f"(ref[0]), "f"(cur.fx[0]), "n"(PB), "n"(PB + 4));
                } else {
                    static_assert(C == 2, "fused kernel: 1 or 2 columns per thread");
                    asm volatile(
                        "{\n\t.reg .pred p;\n\t.reg .f32 s0, s1, s2, s3;\n\t"
                        "setp.lt.s32 p, %6, 0;\n\t"
                        "@!p bra.uni SKIP_%=;\n\t"
                        "add.u32 %0, %0, %11;\n\t"
                        "add.u32 %3, %3, %11;\n\t"
                        "ld.shared.f32 s0, [%0+%11];\n\t"
                        "ld.shared.f32 s1, [%0+%12];\n\t"
                        "ld.shared.f32 s2, [%3+%11];\n\t"
                        "ld.shared.f32 s3, [%3+%12];\n\t"
                        "mov.f32 %1, %2;\n\t"
                        "mov.f32 %4, %5;\n\t"
                        "sub.f32 s1, s1, s0;\n\t"
                        "sub.f32 s3, s3, s2;\n\t"
                        "sub.f32 s0, s0, %7;\n\t"
                        "sub.f32 s2, s2, %9;\n\t"
                        "fma.rn.f32 %2, %8, s1, s0;\n\t"
                        "fma.rn.f32 %5, %10, s3, s2;\n\t"
                        "SKIP_%=:\n\t}"
                        : "+r"(tp[0]), "+f"(T[0]), "+f"(B[0]), "+r"(tp[1]), "+f"(T[1]), "+f"(B[1])
                        : "r"(__float_as_int(code)), "f"(ref[0]), "f"(cur.fx[0]), "f"(ref[1]), "f"(cur.fx[1]),
                          "n"(PB), "n"(PB + 4));
                }
            }
            const float fy = fabsf(code), omfy = 1.0f - fy;
#pragma unroll
            for (int c = 0; c < C; ++c) acc[c][i] = fmaf(fy, B[c], fmaf(omfy, T[c], acc[c][i]));
        }
        cur = nxt;
        __syncthreads();                                   // every warp is done with stage a % NS
        if (warp == 0 && a + NS < nact) issue(a + NS);
    }
    __syncthreads();                                       // tiles are dead: shared memory becomes the exchange buffer

    // ---- phase B: image formation, one (subaperture row, column slot) round at a time ----
    const float scale = (float)sp.scale;
    const int g = tid / n, b = tid - g * n;                // subaperture in round, column in subaperture
    const size_t set = (size_t)k * A.n_sel + si;
    float2* xs = xch + (size_t)g * K::SUB_STRIDE;
    bool first_round = true;
#pragma unroll
    for (int h = 0; h < R2; ++h) {
#pragma unroll
        for (int c = 0; c < C; ++c) {
            const int gs = c * K::GS + g;                  // subaperture within the item
            const int q = it.q0 + gs, p = it.p + h;
            const int sa = p * A.n_sub + q;
            const bool active = gs < it.cnt && p < A.n_sub && A.valid[sa] != 0;
            if (!first_round) __syncthreads();             // previous round finished reading the exchange buffer
            first_round = false;
            if (__any_sync(0xffffffffu, active)) {
                float2 e[n];
                const float* ap = A.amp + (size_t)(p * n) * N + (size_t)q * n + b;
#pragma unroll
                for (int i = 0; i < n; ++i) {
                    const float Am = active ? __ldg(ap + (size_t)i * N) : 0.0f;
                    float s, co;
                    sincosf(acc[c][h * n + i] * scale, &s, &co);
                    e[i] = make_float2(Am * co, Am * s);
                }
                dft_half_padded<M>(e, [&](auto ki, const float2 v) {
                    constexpr int kk = decltype(ki)::value;
                    xs[kk * K::XP + b] = v;                // column FFT result: T[k][b]
                });
            }
            __syncthreads();
            if (!__any_sync(0xffffffffu, active)) continue;
            // rows k = b and k = b + n of this subaperture
            float pixv[2][P];
            int cbase = 0;
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
            constexpr int NPIX = P / BETA;                 // pixels kept per row after the exchange
            // detector rows of this thread: r = (b + hh n) / BETA ; columns cbase .. cbase + NPIX - 1
            float s = 0.0f, mx = 0.0f, my = 0.0f;
#pragma unroll
            for (int hh = 0; hh < 2; ++hh) {
                const int r = (b + hh * n) / BETA;
#pragma unroll
                for (int i = 0; i < NPIX; ++i) {
                    float v = pixv[hh][i];
                    const int col = cbase + i;
                    if (NOISE) {
                        if (active) v = noisy_pixel(v, A.nz, (uint32_t)(r * P + col), (uint32_t)sa, (uint32_t)src_index,
                                                    (uint32_t)(A.step0 + k));
                    }
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
}

// ------------------------------------------------------------------------------------------------
// host side
template <int M, int G, int C, int R2>
static cudaError_t launch_variant(ao_geometry* g, const WfsH& w, const FusedArgs& a, int n_items, int n_steps,
                                  cudaStream_t st)
{
    using K = FusedCfg<M, G, C, R2>;
    auto kern = a.nz.on ? k_fused<M, G, C, R2, true> : k_fused<M, G, C, R2, false>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)K::SMEM);
    if (e != cudaSuccess) return e;
    for (int k0 = 0; k0 < n_steps; k0 += 65535) {
        const int ks = n_steps - k0 < 65535 ? n_steps - k0 : 65535;
        FusedArgs b = a;
        b.step0 = a.step0 + k0;
        const size_t set0 = (size_t)k0 * a.n_sel, nsa = (size_t)w.n_sub * w.n_sub;
        if (a.images) b.images = a.images + set0 * nsa * w.P * w.P;
        if (a.slopes) b.slopes = a.slopes + set0 * 2 * nsa;
        kern<<<dim3(n_items, a.n_sel, ks), K::NT, K::SMEM, st>>>(b);
        g->launches++;
        if ((e = cudaGetLastError()) != cudaSuccess) return e;
    }
    return cudaSuccess;
}

// Tile shape of the fused kernel per FFT size: G subapertures wide, R2 subaperture rows tall.
void fused_tile_shape(int M, int* G, int* R2)
{
    if (M == 32) { *G = 16; *R2 = 2; }
    else if (M == 16) { *G = 32; *R2 = 2; }
    else { *G = 0; *R2 = 0; }
}

bool fused_supported(const ao_geometry* g, const WfsH& w)
{
    if (!(w.M == 16 || w.M == 32) || w.n * 2 != w.M || w.P != 8 || w.beta * w.P != w.M) return false;
    if (w.fused_items == nullptr || w.n_fused_items == 0) return false;
    int G, R2; fused_tile_shape(w.M, &G, &R2);
    for (int s : w.grp.src) {
        const SourceP& sp = g->sources[s];
        for (const LayerP& lp : g->layers) {
            if (!(lp.height < sp.H)) continue;
            const double du = (1.0 - lp.height * sp.inv_H) * sp.d * lp.inv_pitch;
            if (!(du > 0.0) || du > 1.0) return false;            // the row march assumes 0 < du <= 1
            if (lp.S % 4 != 0) return false;                       // 16-byte aligned rows for the bulk copies
            if (lp.S < G * w.n + 8 || lp.S < R2 * w.n + 2) return false;
        }
    }
    return true;
}

cudaError_t launch_fused(ao_geometry* g, const WfsH& w, int64_t step0, int n_steps, double dt,
                         const NoiseP& noise, float* images, float* slopes, cudaStream_t st)
{
    if (!fused_supported(g, w)) return cudaErrorNotSupported;
    const size_t n_sel = w.grp.src.size(), nsa = (size_t)w.n_sub * w.n_sub;
    cudaError_t e;
    // invalid subapertures are never scheduled: zero-fill the outputs first
    if (images && (e = cudaMemsetAsync(images, 0, sizeof(float) * n_steps * n_sel * nsa * w.P * w.P, st)) != cudaSuccess) return e;
    if (slopes && (e = cudaMemsetAsync(slopes, 0, sizeof(float) * n_steps * n_sel * 2 * nsa, st)) != cudaSuccess) return e;
    FusedArgs a;
    a.layers = g->d_layers; a.n_layers = (int)g->layers.size();
    a.srcs = g->d_sources; a.sel = w.grp.d_src; a.n_sel = (int)n_sel;
    a.items = (const WorkItem*)w.fused_items; a.amp = w.d_amp; a.valid = w.d_valid; a.n_sub = w.n_sub;
    a.step0 = step0; a.dt = dt;
    a.norm = (float)(1.0 / ((double)w.M * w.M * (double)w.n * w.n));
    a.nz = noise; a.images = images; a.slopes = slopes;
    if (w.M == 32) return launch_variant<32, 16, 2, 2>(g, w, a, w.n_fused_items, n_steps, st);
    return launch_variant<16, 32, 2, 2>(g, w, a, w.n_fused_items, n_steps, st);
}

}  // namespace ao
