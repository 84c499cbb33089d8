// k_fft_big.cu -- two-pass HBM/L2 FFT for the large transforms: the science PSF (section 2.8,
// reading O7) and the NGS low-order Shack-Hartmann sensors with FFT > 64 (readings O3/O4).
//
// Both passes run register-resident Stockham FFTs: a thread holds 16 complex points, a transform of
// M = 2^LOGM points is T = M/16 threads and two or three radix-16/16/(M/256) passes; points change hands
// between passes through shared memory padded by one slot every 16 (conflict-free reads and writes);
// the first pass reads global memory directly and the last one writes it, in natural order.
//
// Pass 1 (k_big_rows): the n non-zero input rows only (pruning).  Builds E = A exp(i phi) pre[a] pre[b]
//   on the fly (pre carries the centring: (-1)^a for the pixel-centred PSF, exp(+i pi (M-1) a/M) for the
//   half-pixel-centred SH), transforms the zero-padded row and writes it to the scratch T[batch][a][m].
//   A CTA of 256 threads handles 256/T rows.
// Pass 2 (k_big_cols): a CTA of T*C threads transforms C adjacent columns (thread = (point group, column),
//   column fastest, so that global reads are C*8-byte row segments and the shared-memory image is
//   column-interleaved), takes |.|^2 and
//   - PSF: accumulates the steps of a chunk in registers and adds them to the long exposure once;
//   - SH: sums the beta x beta detector bins (C = beta: one detector column per CTA).
// The scratch of a chunk is sized near the L2 capacity, but ncu --cache-control none shows that most of it is written
// back to DRAM before the column pass reads it (profiles/r2_big_fft_l2.md): the passes are latency-bound, not DRAM-bound.
#include <algorithm>
#include <mutex>
#include <string>

#include "fft_big.cuh"

namespace ao {

struct BigRowArgs {
    const float* phase; long long step_stride; const long long* off; int n_sel;
    const float* amp; const uint8_t* valid; int n_sub, n;
    const float2* tw; const float2* pre; float2* T;
};

// Pass 1.  grid (ceil(n / rows per CTA), batch), batch index b = (step * n_sel + si) * n_sub^2 + sa.
template <int LOGM>
__global__ void __launch_bounds__(256, 4)
k_big_rows(const BigRowArgs A)
{
    using K = BigCfg<LOGM>;
    constexpr int M = K::M, T = K::T, RPC = 256 / T;
    extern __shared__ float4 smem_raw[];
    float2* sm = reinterpret_cast<float2*>(smem_raw);
    const int tid = threadIdx.x, r = tid / T, tb = tid - r * T;
    const int n = A.n, nsa = A.n_sub * A.n_sub;
    const long long b = blockIdx.y;
    const int sa = (int)(b % nsa);
    const long long set = b / nsa;
    const int si = (int)(set % A.n_sel);
    const long long k = set / A.n_sel;
    if (A.valid && !A.valid[sa]) return;                                   // CTA-uniform
    const int a = blockIdx.x * RPC + r;
    const bool row_on = a < n;
    const int p = sa / A.n_sub, q = sa - p * A.n_sub, N = A.n_sub * n;
    const size_t rowoff = (size_t)(p * n + (row_on ? a : 0)) * N + (size_t)q * n;
    const float* ph = A.phase + (size_t)k * A.step_stride + A.off[si] + rowoff;
    const float* am = A.amp + rowoff;
    const float2 pa = row_on ? A.pre[a] : make_float2(0.0f, 0.0f);
    float2* out = A.T + ((size_t)b * n + (row_on ? a : 0)) * M;
    // all global loads of the thread's 16 input points are issued before the first use (predicated, no branch): the row
    // pass used to wait for each load in turn (30 % of its stall samples)
    float ph_r[16], am_r[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) {
        const int i = tb + k * (M / 16);
        const bool on = row_on && i < n;
        ph_r[k] = on ? __ldg(ph + i) : 0.0f;
        am_r[k] = on ? __ldg(am + i) : 0.0f;
    }
    big_fft<LOGM>(tb, sm, 1, r * K::PADM, A.tw,
        [&](int i) {
            const int k = (i - tb) >> (LOGM - 4);                  // first pass: point i = tb + k M/16 (folds to a constant)
            float2 v = make_float2(0.0f, 0.0f);
            if (row_on && i < n) {
                float s, c;
                sincos_reduced(ph_r[k], &s, &c);
                const float2 w = cmulf(pa, __ldg(A.pre + i));
                v = cmulf(make_float2(am_r[k] * c, am_r[k] * s), w);
            }
            return v;
        },
        [&](int i, const float2 x, int) { if (row_on) out[i] = x; });
}

struct BigColArgs {
    const float2* T; const uint8_t* valid; int nsa, n, C;
    const float2* tw; float norm;
    int beta, P, k0;                  // SH: detector window
    int n_dir, ks, accumulate;        // PSF: directions, steps in the chunk, += or =
    float* out;
};

// Pass 2.  MODE 0 (PSF): grid (M / C, n_dir); the CTA loops over the ks steps of the chunk.
//          MODE 1 (SH):  grid (P, batch), C = beta, columns k0 + g beta .. of the detector window.
// CT: columns per CTA as a compile-time constant (0 = run-time A.C): with it every shared-memory index of the
// Stockham passes is a per-thread base plus an immediate instead of a multiply per point.
template <int LOGM, int MODE, int CT>
__global__ void __launch_bounds__(MODE == 0 ? 512 : 1024)
k_big_cols(const BigColArgs A)
{
    using K = BigCfg<LOGM>;
    constexpr int M = K::M;
    extern __shared__ float4 smem_raw[];
    float2* sm = reinterpret_cast<float2*>(smem_raw);
    const int tid = threadIdx.x, C = CT ? CT : A.C, tb = tid / C, c = tid - tb * C;
    const int n = A.n, g = blockIdx.x;
    const long long b = blockIdx.y;
    if (MODE == 0) {
        const int m0 = g * C;
        float acc[16];
#pragma unroll
        for (int i = 0; i < 16; ++i) acc[i] = 0.0f;
        for (int k = 0; k < A.ks; ++k) {
            const float2* Tb = A.T + ((size_t)(k * A.n_dir + b) * n) * M + m0 + c;
            big_fft<LOGM>(tb, sm, C, c, A.tw,
                [&](int i) { return i < n ? ldg_stream(Tb + (size_t)i * M) : make_float2(0.0f, 0.0f); },
                [&](int, const float2 x, int slot) { acc[slot] = fmaf(x.x, x.x, fmaf(x.y, x.y, acc[slot])); });
            __syncthreads();                                  // the next step overwrites the exchange buffer
        }
        float* o = A.out + (size_t)b * M * M + m0 + c;
        // replay the index arithmetic of the last pass to place the 16 accumulators
        constexpr int RL = K::R2 == 1 ? K::R1 : K::R2, NSL = K::R2 == 1 ? 16 : 256, Q = 16 / RL;
#pragma unroll
        for (int q = 0; q < Q; ++q) {
            const int bb = tb + q * K::T;
            const int o0 = (bb / NSL) * (NSL * RL) + (bb & (NSL - 1));
#pragma unroll
            for (int kk = 0; kk < RL; ++kk) {
                const size_t gi = (size_t)(o0 + kk * NSL) * M;
                const float I = acc[q * RL + kk] * A.norm;
                o[gi] = A.accumulate ? o[gi] + I : I;
            }
        }
    } else {
        const int sa = (int)(b % A.nsa);
        if (A.valid && !A.valid[sa]) {
            for (int r = tid; r < A.P; r += blockDim.x) A.out[((size_t)b * A.P + r) * A.P + g] = 0.0f;
            return;
        }
        const int m0 = A.k0 + g * A.beta;
        const float2* Tb = A.T + (size_t)b * n * M + m0 + c;
        float I[16];
        big_fft<LOGM>(tb, sm, C, c, A.tw,
            [&](int i) { return i < n ? ldg_stream(Tb + (size_t)i * M) : make_float2(0.0f, 0.0f); },
            [&](int, const float2 x, int slot) { I[slot] = fmaf(x.x, x.x, x.y * x.y); });
        __syncthreads();                                      // every thread has finished reading the exchange buffer
        // intensities to shared memory as Ib[i][c] (replaying the index arithmetic of the last pass), then one
        // warp per detector pixel sums its beta x beta block, which is beta * C contiguous floats
        float* Ib = reinterpret_cast<float*>(sm);
        constexpr int RL = K::R2 == 1 ? K::R1 : K::R2, NSL = K::R2 == 1 ? 16 : 256, Q = 16 / RL;
#pragma unroll
        for (int q = 0; q < Q; ++q) {
            const int bb = tb + q * K::T;
            const int o0 = (bb / NSL) * (NSL * RL) + (bb & (NSL - 1));
#pragma unroll
            for (int kk = 0; kk < RL; ++kk) Ib[(o0 + kk * NSL) * C + c] = I[q * RL + kk];
        }
        __syncthreads();
        const int lane = tid & 31, warp = tid >> 5, nw = (int)(blockDim.x >> 5), span = A.beta * C;
        if (span == 64) {
            // 8 x 8 bins (the NGS sensors): a pixel is 64 contiguous floats; 8 threads per pixel, two LDS.128 each (the 8
            // lanes of a quarter-warp read 8 consecutive float4: conflict-free), three shuffles.  The generic loop below
            // was 42 % of this kernel's instructions.
            const int sub = tid & 7;
            for (int r = tid >> 3; r < A.P; r += (int)(blockDim.x >> 3)) {
                const float4* src = reinterpret_cast<const float4*>(Ib + (size_t)(A.k0 + r * A.beta) * C);
                const float4 a = src[sub], b4 = src[8 + sub];
                float s = ((a.x + a.y) + (a.z + a.w)) + ((b4.x + b4.y) + (b4.z + b4.w));
                s += __shfl_xor_sync(0xffffffffu, s, 1);
                s += __shfl_xor_sync(0xffffffffu, s, 2);
                s += __shfl_xor_sync(0xffffffffu, s, 4);
                if (sub == 0) A.out[((size_t)b * A.P + r) * A.P + g] = s * A.norm;
            }
            return;
        }
        for (int r = warp; r < A.P; r += nw) {
            const float* src = Ib + (size_t)(A.k0 + r * A.beta) * C;
            float s = 0.0f;
            for (int e = lane; e < span; e += 32) s += src[e];
            s = warp_sum(s);
            if (lane == 0) A.out[((size_t)b * A.P + r) * A.P + g] = s * A.norm;
        }
    }
}

// ---- M = 64: the whole subaperture in one CTA -------------------------------------------------
// One CTA of 256 threads per (step, source, subaperture): both passes of the 64 x 64 transform and the binning
// stay in shared memory (no HBM scratch; the two-pass kernels above would move 16 KB per subaperture frame twice).
// Pass A: the n non-zero rows, 4 threads per 64-point Stockham transform (64 transforms per CTA-wide call);
// pass B: the 64 columns the same way, |.|^2 into shared memory; then beta x beta binning, 4 threads per pixel.
struct MidArgs {
    const float* phase; long long step_stride; const long long* off; int n_sel;
    const float* amp; const uint8_t* valid; int n_sub, n;
    const float2* tw; const float2* pre;
    int beta, P, k0; float norm;
    float* out;                                            // [batch][P][P]
};

__global__ void __launch_bounds__(256, 4)
k_sh_mid64(const MidArgs A)
{
    using K = BigCfg<6>;
    constexpr int M = 64, T = K::T, NTR = 256 / T, TP = M + 1;     // 64 transforms per pass, padded pitch
    extern __shared__ float4 smem_raw[];
    float2* sm = reinterpret_cast<float2*>(smem_raw);                // exchange buffer of the passes: [64][PADM]
    float2* Tm = sm + NTR * K::PADM;                                 // row-pass output [n <= 64][TP] (n <= 32 used)
    float* Ib = reinterpret_cast<float*>(Tm);                        // |.|^2 [M][TP], aliases Tm after pass B's loads
    const int tid = threadIdx.x, r = tid / T, tb = tid - r * T;
    const int n = A.n, nsa = A.n_sub * A.n_sub, P = A.P;
    const long long b = blockIdx.x;
    const int sa = (int)(b % nsa);
    const long long set = b / nsa;
    const int si = (int)(set % A.n_sel);
    const long long k = set / A.n_sel;
    float* out = A.out + (size_t)b * P * P;
    if (A.valid && !A.valid[sa]) {                                   // CTA-uniform
        for (int i = tid; i < P * P; i += 256) out[i] = 0.0f;
        return;
    }
    const int p = sa / A.n_sub, q = sa - p * A.n_sub, N = A.n_sub * n;
    {   // pass A: row r of the subaperture (rows >= n are zero and are not transformed: their output is unused)
        const bool row_on = r < n;
        const size_t rowoff = (size_t)(p * n + (row_on ? r : 0)) * N + (size_t)q * n;
        const float* ph = A.phase + (size_t)k * A.step_stride + A.off[si] + rowoff;
        const float* am = A.amp + rowoff;
        const float2 pa = row_on ? A.pre[r] : make_float2(0.0f, 0.0f);
        big_fft<6>(tb, sm, 1, r * K::PADM, A.tw,
            [&](int i) {
                float2 v = make_float2(0.0f, 0.0f);
                if (row_on && i < n) {
                    const float Am = __ldg(am + i);
                    float s, c;
                    sincos_reduced(__ldg(ph + i), &s, &c);
                    v = cmulf(make_float2(Am * c, Am * s), cmulf(pa, __ldg(A.pre + i)));
                }
                return v;
            },
            [&](int i, const float2 x, int) { if (row_on) Tm[r * TP + i] = x; });
    }
    __syncthreads();
    float I[16];
    big_fft<6>(tb, sm, 1, r * K::PADM, A.tw,                         // pass B: column m = r
        [&](int i) { return i < n ? Tm[i * TP + r] : make_float2(0.0f, 0.0f); },
        [&](int, const float2 x, int slot) { I[slot] = fmaf(x.x, x.x, x.y * x.y); });
    __syncthreads();                                                 // every thread has finished reading Tm
    {
        constexpr int RL = K::R1, NSL = 16, Q = 16 / RL;            // index arithmetic of the last pass (two passes)
#pragma unroll
        for (int qq = 0; qq < Q; ++qq) {
            const int bb = tb + qq * T;
            const int o0 = (bb / NSL) * (NSL * RL) + (bb & (NSL - 1));
#pragma unroll
            for (int kk = 0; kk < RL; ++kk) Ib[(o0 + kk * NSL) * TP + r] = I[qq * RL + kk];     // Ib[row k][column m]
        }
    }
    __syncthreads();
    // binning: pixel (pr, pc) sums rows k0 + pr beta .. and columns k0 + pc beta ..; 4 threads per pixel
    const int beta = A.beta, part = tid & 3;
    for (int px = tid >> 2; px < P * P; px += 64) {
        const int pr = px / P, pc = px - pr * P;
        float s = 0.0f;
        for (int e = part; e < beta * beta; e += 4) {
            const int er = e / beta, ec = e - er * beta;
            s += Ib[(A.k0 + pr * beta + er) * TP + A.k0 + pc * beta + ec];
        }
        s += __shfl_xor_sync(0xffffffffu, s, 1);
        s += __shfl_xor_sync(0xffffffffu, s, 2);
        if (part == 0) out[px] = s * A.norm;
    }
}

// ---- host side -------------------------------------------------------------------------------
size_t sh_big_scratch_bytes(const ao_geometry*, const WfsH& w)
{
    if (w.M == 64) return 0;                                  // k_sh_mid64 keeps the whole transform in shared memory
    return sizeof(float2) * (size_t)w.grp.src.size() * w.n_sub * w.n_sub * w.n * w.M;
}

size_t psf_scratch_bytes(const ao_geometry* g)
{
    return sizeof(float2) * g->sci.src.size() * (size_t)g->Np * g->psf_fft;
}

// Steps of the science PSF transformed per launch pair: the column pass sums them in registers, so the
// long exposure is read and written once per chunk; the scratch of a chunk is bounded (64 MB).
int psf_chunk_steps(const ao_geometry* g)
{
    const size_t per = psf_scratch_bytes(g);
    if (per == 0) return 1;
    const size_t budget = (size_t)3 << 29;                   // 1.5 GB of scratch at most
    size_t ks = budget / per;
    if (ks < 1) ks = 1;
    if (ks > 16) ks = 16;
    return (int)ks;
}

static int cols_threads_per_transform(int M) { return M / 16; }

// The SH fast path needs C = beta columns per CTA: a power of two, full warps, at most 1024 threads.
bool sh_big_fast(const WfsH& w)
{
    if (w.M < 64 || w.M > 4096 || (w.M & (w.M - 1))) return false;
    const int T = cols_threads_per_transform(w.M), C = w.beta;
    if (C < 1 || C > 32 || (C & (C - 1))) return false;
    if (T * C < 32 || T * C > 1024 || w.P > 1024) return false;
    return sizeof(float2) * (size_t)C * (w.M + w.M / 16) <= 200 * 1024;
}

template <int LOGM>
static cudaError_t launch_rows_t(const BigRowArgs& a, int n_rows, unsigned batch, cudaStream_t st)
{
    using K = BigCfg<LOGM>;
    constexpr int RPC = 256 / K::T;
    const size_t smem = sizeof(float2) * (size_t)RPC * K::PADM;
    cudaError_t e = cudaFuncSetAttribute(k_big_rows<LOGM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    k_big_rows<LOGM><<<dim3((n_rows + RPC - 1) / RPC, batch), 256, smem, st>>>(a);
    return cudaGetLastError();
}

template <int LOGM, int MODE, int CT>
static cudaError_t launch_cols_ct(const BigColArgs& a, unsigned gx, unsigned gy, cudaStream_t st)
{
    using K = BigCfg<LOGM>;
    const size_t smem = sizeof(float2) * (size_t)a.C * K::PADM;
    cudaError_t e = cudaFuncSetAttribute(k_big_cols<LOGM, MODE, CT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    k_big_cols<LOGM, MODE, CT><<<dim3(gx, gy), K::T * a.C, smem, st>>>(a);
    return cudaGetLastError();
}

template <int LOGM, int MODE>
static cudaError_t launch_cols_t(const BigColArgs& a, unsigned gx, unsigned gy, cudaStream_t st)
{
    constexpr int CFAST = MODE == 0 ? 4 : 8;               // PSF at M >= 512 uses 4 columns, the NGS sensors bin 8 x 8
    if (a.C == CFAST) return launch_cols_ct<LOGM, MODE, CFAST>(a, gx, gy, st);
    return launch_cols_ct<LOGM, MODE, 0>(a, gx, gy, st);
}

#define AO_BIG_DISPATCH(logM, CALL)                                   \
    switch (logM) {                                                   \
        case 6: { constexpr int L = 6; return CALL; }                 \
        case 7: { constexpr int L = 7; return CALL; }                 \
        case 8: { constexpr int L = 8; return CALL; }                 \
        case 9: { constexpr int L = 9; return CALL; }                 \
        case 10: { constexpr int L = 10; return CALL; }               \
        case 11: { constexpr int L = 11; return CALL; }               \
        case 12: { constexpr int L = 12; return CALL; }               \
        default: return cudaErrorNotSupported;                        \
    }

static cudaError_t launch_rows(int logM, const BigRowArgs& a, int n_rows, unsigned batch, cudaStream_t st)
{
    AO_BIG_DISPATCH(logM, launch_rows_t<L>(a, n_rows, batch, st))
}
static cudaError_t launch_cols_psf(int logM, const BigColArgs& a, unsigned gx, unsigned gy, cudaStream_t st)
{
    AO_BIG_DISPATCH(logM, (launch_cols_t<L, 0>(a, gx, gy, st)))
}
static cudaError_t launch_cols_sh(int logM, const BigColArgs& a, unsigned gx, unsigned gy, cudaStream_t st)
{
    AO_BIG_DISPATCH(logM, (launch_cols_t<L, 1>(a, gx, gy, st)))
}

cudaError_t launch_sh_big_generic(ao_geometry* g, const WfsH& w, const float* phase, bool api_layout,
                                  long long step_stride, int n_steps, float2* scratch, float* images,
                                  cudaStream_t st);

cudaError_t launch_sh_big(ao_geometry* g, const WfsH& w, const float* phase, bool api_layout,
                          long long step_stride, int n_steps, float2* scratch, size_t scratch_bytes, float* images,
                          cudaStream_t st)
{
    const int n_sel = (int)w.grp.src.size(), nsa = w.n_sub * w.n_sub;
    if (n_sel == 0 || n_steps <= 0) return cudaSuccess;
    cudaError_t e;
    if (w.M == 64) {      // whole subaperture per CTA
        const size_t smem = sizeof(float2) * (size_t)(64 * BigCfg<6>::PADM) +
                            std::max(sizeof(float2) * (size_t)w.n * 65, sizeof(float) * (size_t)64 * 65);
        if ((e = cudaFuncSetAttribute(k_sh_mid64, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)) != cudaSuccess) return e;
        MidArgs m;
        m.phase = phase; m.step_stride = step_stride; m.off = api_layout ? w.grp.d_off_api : w.grp.d_off_stage;
        m.n_sel = n_sel; m.amp = w.d_amp; m.valid = w.d_valid; m.n_sub = w.n_sub; m.n = w.n;
        m.tw = w.d_twf; m.pre = w.d_pre; m.beta = w.beta; m.P = w.P; m.k0 = (w.M - w.beta * w.P) / 2;
        m.norm = (float)(1.0 / ((double)w.M * w.M * (double)w.n * w.n));
        const long long total = (long long)n_steps * n_sel * nsa;
        const long long chunk = 0x7fffffffLL / ((long long)n_sel * nsa) * ((long long)n_sel * nsa);
        for (long long b0 = 0; b0 < total; b0 += chunk) {
            const long long nb = total - b0 < chunk ? total - b0 : chunk;
            m.phase = phase + (size_t)(b0 / ((long long)n_sel * nsa)) * step_stride;
            m.out = images + (size_t)b0 * w.P * w.P;
            k_sh_mid64<<<(unsigned)nb, 256, smem, st>>>(m);
            g->launches++;
            if ((e = cudaGetLastError()) != cudaSuccess) return e;
        }
        return cudaSuccess;
    }
    if (!sh_big_fast(w)) return launch_sh_big_generic(g, w, phase, api_layout, step_stride, n_steps, scratch, images, st);
    const unsigned batch = (unsigned)(n_sel * nsa);
    // as many steps per launch pair as the scratch holds (at most 4 and 96 MB: two steps of the NGS sensors measured best)
    const size_t per_step = sh_big_scratch_bytes(g, w);
    int kb = per_step ? (int)std::min<size_t>(8, scratch_bytes / per_step) : 1;
    if (kb < 1) kb = 1;
    while (kb > 1 && (size_t)kb * batch > 65535u) --kb;    // the batch is gridDim.y (ao_geometry_create bounds one step)
    for (int k = 0; k < n_steps; k += kb) {
        const int kn = n_steps - k < kb ? n_steps - k : kb;
        BigRowArgs r;
        r.phase = phase + (size_t)k * step_stride; r.step_stride = step_stride;
        r.off = api_layout ? w.grp.d_off_api : w.grp.d_off_stage; r.n_sel = n_sel;
        r.amp = w.d_amp; r.valid = w.d_valid; r.n_sub = w.n_sub; r.n = w.n;
        r.tw = w.d_twf; r.pre = w.d_pre; r.T = scratch;
        if ((e = launch_rows(w.logM, r, w.n, batch * (unsigned)kn, st)) != cudaSuccess) return e;
        g->launches++;
        BigColArgs c;
        c.T = scratch; c.valid = w.d_valid; c.nsa = nsa; c.n = w.n; c.C = w.beta; c.tw = w.d_twf;
        c.norm = (float)(1.0 / ((double)w.M * w.M * (double)w.n * w.n));
        c.beta = w.beta; c.P = w.P; c.k0 = (w.M - w.beta * w.P) / 2;
        c.n_dir = 1; c.ks = 1; c.accumulate = 0;
        c.out = images + (size_t)k * batch * w.P * w.P;
        if ((e = launch_cols_sh(w.logM, c, (unsigned)w.P, batch * (unsigned)kn, st)) != cudaSuccess) return e;
        g->launches++;
    }
    return cudaSuccess;
}

// Science PSF of `ks` consecutive steps (phase of step j at phase + j * step_stride), summed and then
// added to (accumulate != 0) or stored in psf.  ks <= psf_chunk_steps(g): the scratch holds ks steps.
cudaError_t launch_psf(ao_geometry* g, const float* phase, bool api_layout, long long step_stride,
                       int ks, float2* scratch, float* psf, int accumulate, cudaStream_t st)
{
    const int n_dir = (int)g->sci.src.size(), M = g->psf_fft;
    if (n_dir == 0 || ks <= 0) return cudaSuccess;
    cudaError_t e;
    BigRowArgs r;
    r.phase = phase; r.step_stride = step_stride;
    r.off = api_layout ? g->sci.d_off_api : g->sci.d_off_stage; r.n_sel = n_dir;
    r.amp = g->d_pupil_amp; r.valid = nullptr; r.n_sub = 1; r.n = g->Np;
    r.tw = g->d_psf_tw; r.pre = g->d_psf_pre; r.T = scratch;
    if ((e = launch_rows(g->psf_log, r, g->Np, (unsigned)(ks * n_dir), st)) != cudaSuccess) return e;
    g->launches++;
    const int T = cols_threads_per_transform(M);
    int C = 4;
    while (T * C < 128) C *= 2;                              // small transforms: keep at least 4 warps per CTA
    while (T * C > 512) C /= 2;                              // launch bound of the PSF column pass
    BigColArgs c;
    c.T = scratch; c.valid = nullptr; c.nsa = 1; c.n = g->Np; c.C = C; c.tw = g->d_psf_tw;
    c.norm = g->sumA2 > 0 ? (float)(1.0 / ((double)M * M * g->sumA2)) : 0.0f;
    c.beta = 1; c.P = 1; c.k0 = 0; c.n_dir = n_dir; c.ks = ks; c.accumulate = accumulate; c.out = psf;
    if ((e = launch_cols_psf(g->psf_log, c, (unsigned)(M / C), (unsigned)n_dir, st)) != cudaSuccess) return e;
    g->launches++;
    return cudaSuccess;
}

}  // namespace ao

// ---- ao_psf_static: the science PSF of one direction with no allocation of any kind ----------------------------
// For callers that cannot call cudaMalloc (CUDA graph capture, tight serving loops, harnesses that forbid it) and
// therefore cannot lend a workspace either: the row pass's intermediate T[Np][M] lives in a file-scope device array
// of AO_PSF_STATIC_MAX_BYTES (16 MiB, held by every GPU that loads the library until the process exits).  Same two
// kernels as ao_psf (k_big_rows, k_big_cols<MODE 0>), one launch pair per step, one direction per call.
// In host code `g_psf_static_scratch` is only a stand-in for the symbol: its device address is looked up once per
// device with cudaGetSymbolAddress (that device current) and kept in g_psf_static_ptr[device].
using namespace ao;

static __device__ __align__(256) float2 g_psf_static_scratch[AO_PSF_STATIC_MAX_BYTES / sizeof(float2)];

static constexpr int kMaxDevices = 64;
static float2* g_psf_static_ptr[kMaxDevices];             // zero-initialised; written once per device
static std::mutex g_psf_static_mutex;

static cudaError_t psf_static_scratch(int device, float2** out)
{
    std::lock_guard<std::mutex> lock(g_psf_static_mutex);
    if (!g_psf_static_ptr[device]) {
        void* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_psf_static_scratch);   // the calling thread's current device
        if (e != cudaSuccess) return e;
        g_psf_static_ptr[device] = static_cast<float2*>(p);
    }
    *out = g_psf_static_ptr[device];
    return cudaSuccess;
}

extern "C" int ao_psf_static(ao_geometry* g, int direction, const float* phase_dev, int n_steps, float* psf_dev,
                             int accumulate, void* cuda_stream)
{
    if (!g || !phase_dev || !psf_dev) { set_error("ao_psf_static: NULL argument"); return AO_ERR_INVALID_ARG; }
    const int n_dir = (int)g->sci.src.size(), M = g->psf_fft;
    if (n_dir == 0 || M == 0) { set_error("ao_psf_static: no science direction / psf_fft == 0"); return AO_ERR_INVALID_ARG; }
    if (direction < 0 || direction >= n_dir || n_steps < 0) {
        set_error("ao_psf_static: direction out of range or n_steps < 0"); return AO_ERR_INVALID_ARG;
    }
    const size_t need = sizeof(float2) * (size_t)g->Np * M;
    if (need > (size_t)AO_PSF_STATIC_MAX_BYTES) {
        set_error("ao_psf_static: pupil n * psf_fft * 8 = " + std::to_string(need) + " bytes exceeds the static scratch of " +
                  std::to_string((size_t)AO_PSF_STATIC_MAX_BYTES) + " bytes (AO_PSF_STATIC_MAX_BYTES): use ao_psf with a workspace");
        return AO_ERR_UNSUPPORTED;
    }
    if (g->device < 0 || g->device >= kMaxDevices) { set_error("ao_psf_static: device ordinal beyond 63"); return AO_ERR_UNSUPPORTED; }
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess && dev != g->device) e = cudaSetDevice(g->device);
    if (e == cudaSuccess) e = cudaPeekAtLastError();
    float2* scratch = nullptr;
    if (e == cudaSuccess) e = psf_static_scratch(g->device, &scratch);
    if (e != cudaSuccess) { set_error(std::string("ao_psf_static: ") + cudaGetErrorString(e)); return AO_ERR_CUDA; }
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    if (n_steps == 0) {
        if (!accumulate) e = cudaMemsetAsync(psf_dev, 0, sizeof(float) * (size_t)M * M, st);
        if (e != cudaSuccess) { set_error(std::string("ao_psf_static: memset: ") + cudaGetErrorString(e)); return AO_ERR_CUDA; }
        return AO_OK;
    }
    const int T = cols_threads_per_transform(M);
    int C = 4;
    while (T * C < 128) C *= 2;
    while (T * C > 512) C /= 2;
    for (int k = 0; k < n_steps && e == cudaSuccess; ++k) {
        // the row pass writes every element of T[Np][M] the column pass reads: nothing has to start at zero
        BigRowArgs r;
        r.phase = phase_dev + (size_t)k * g->phase_elems_per_step; r.step_stride = g->phase_elems_per_step;
        r.off = g->sci.d_off_api + direction; r.n_sel = 1;
        r.amp = g->d_pupil_amp; r.valid = nullptr; r.n_sub = 1; r.n = g->Np;
        r.tw = g->d_psf_tw; r.pre = g->d_psf_pre; r.T = scratch;
        e = launch_rows(g->psf_log, r, g->Np, 1u, st);
        if (e != cudaSuccess) break;
        g->launches++;
        BigColArgs c;
        c.T = scratch; c.valid = nullptr; c.nsa = 1; c.n = g->Np; c.C = C; c.tw = g->d_psf_tw;
        c.norm = g->sumA2 > 0 ? (float)(1.0 / ((double)M * M * g->sumA2)) : 0.0f;
        c.beta = 1; c.P = 1; c.k0 = 0; c.n_dir = 1; c.ks = 1; c.accumulate = (accumulate || k > 0) ? 1 : 0; c.out = psf_dev;
        e = launch_cols_psf(g->psf_log, c, (unsigned)(M / C), 1u, st);
        if (e == cudaSuccess) g->launches++;
    }
    if (e != cudaSuccess) { set_error(std::string("ao_psf_static: launch: ") + cudaGetErrorString(e)); return AO_ERR_CUDA; }
    return AO_OK;
}
