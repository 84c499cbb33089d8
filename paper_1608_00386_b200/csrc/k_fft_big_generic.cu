// k_fft_big_generic.cu -- fallback two-pass HBM FFT for large transforms whose shape is outside the fast
// path of k_fft_big.cu (bin factor not a power of two, or too many threads per detector column).
// PAPER.md:86 (science PSF, reading O7) and the NGS Shack-Hartmann with FFT > 64 (readings O3/O4).
//
// Pass 1 (k_big_rows_generic): one CTA per non-zero input row: E = A exp(i phi) pre[a] pre[b], zero-padded
//   radix-2 DIF FFT in shared memory, natural-order row written to the scratch T[batch][a][m].
// Pass 2 (k_big_cols_generic): one CTA per group of C adjacent columns: column FFTs in shared memory,
//   |.|^2 * norm, PSF accumulation (C = 8) or beta x beta binning (C = beta).
#include "ao_device.cuh"

namespace ao {

// In-place radix-2 decimation-in-frequency FFT of `nfft` interleaved transforms of length M held
// in shared memory as x[f*M + i].  Natural-order input, bit-reversed output.  tw[k] = exp(-2 pi i k/M).
__device__ __forceinline__ void fft_dif_smem(float2* x, int M, int logM, int nfft,
                                             const float2* __restrict__ tw, int tid, int nt)
{
    const int halfM = M >> 1, total = nfft * halfM;
    for (int s = 0; s < logM; ++s) {
        const int half = halfM >> s;                 // M/2, M/4, ..., 1
        for (int t = tid; t < total; t += nt) {
            const int f = t / halfM, b = t - f * halfM;
            const int pos = b & (half - 1), grp = b >> (logM - 1 - s);
            const int i = f * M + grp * 2 * half + pos;
            const float2 a = x[i], c = x[i + half];
            const float2 w = __ldg(tw + (pos << s));
            const float dr = a.x - c.x, di = a.y - c.y;
            x[i] = make_float2(a.x + c.x, a.y + c.y);
            x[i + half] = make_float2(dr * w.x - di * w.y, dr * w.y + di * w.x);
        }
        __syncthreads();
    }
}

__global__ void __launch_bounds__(256)
k_big_rows_generic(const float* __restrict__ phase, long long step_stride, const long long* __restrict__ off,
           int n_sel, const float* __restrict__ amp, const uint8_t* __restrict__ valid, int n_sub, int n,
           int M, int logM, const float2* __restrict__ tw, const float2* __restrict__ pre,
           float2* __restrict__ T)
{
    extern __shared__ float4 smem_raw[];
    float2* x = reinterpret_cast<float2*>(smem_raw);
    const int a = blockIdx.x, tid = threadIdx.x, nt = blockDim.x;
    const int nsa = n_sub * n_sub;
    const long long b = blockIdx.y;
    const int sa = (int)(b % nsa);
    const long long set = b / nsa;
    const int si = (int)(set % n_sel);
    const long long k = set / n_sel;
    if (valid && !valid[sa]) return;
    const int p = sa / n_sub, q = sa - p * n_sub, N = n_sub * n;
    const float* ph = phase + (size_t)k * step_stride + off[si] + (size_t)(p * n + a) * N + q * n;
    const float* am = amp + (size_t)(p * n + a) * N + q * n;
    const float2 pa = pre[a];
    for (int i = tid; i < M; i += nt) {
        float2 v = make_float2(0.0f, 0.0f);
        if (i < n) {
            const float A = am[i];
            float s, c;
            sincosf(ph[i], &s, &c);
            const float2 pb = pre[i];
            const float wr = pa.x * pb.x - pa.y * pb.y, wi = pa.x * pb.y + pa.y * pb.x;
            v = make_float2(A * (c * wr - s * wi), A * (c * wi + s * wr));
        }
        x[i] = v;
    }
    __syncthreads();
    fft_dif_smem(x, M, logM, 1, tw, tid, nt);
    float2* out = T + ((size_t)b * n + a) * M;
    for (int m = tid; m < M; m += nt) out[m] = x[__brev((unsigned)m) >> (32 - logM)];
}

// mode 0: PSF (out[dir][k][m] (+)= I), mode 1: SH (images[b][r][g] = binned I)
template <int MODE>
__global__ void __launch_bounds__(256)
k_big_cols_generic(const float2* __restrict__ T, const uint8_t* __restrict__ valid, int nsa, int n, int M, int logM,
           int C, const float2* __restrict__ tw, float norm, int beta, int P, int k0, int accumulate,
           float* __restrict__ out)
{
    extern __shared__ float4 smem_raw[];
    float2* x = reinterpret_cast<float2*>(smem_raw);            // [C][M]
    const int tid = threadIdx.x, nt = blockDim.x;
    const long long b = blockIdx.y;
    const int g = blockIdx.x;
    const int m0 = (MODE == 0) ? g * C : k0 + g * beta;
    if (MODE == 1 && valid && !valid[(int)(b % nsa)]) {
        for (int r = tid; r < P; r += nt) out[((size_t)b * P + r) * P + g] = 0.0f;
        return;
    }
    const float2* Tb = T + (size_t)b * n * M;
    for (int i = tid; i < C * M; i += nt) {
        const int a = i / C, c = i - a * C;                     // c fastest: C*8-byte segments
        x[c * M + a] = (a < n) ? Tb[(size_t)a * M + m0 + c] : make_float2(0.0f, 0.0f);
    }
    __syncthreads();
    fft_dif_smem(x, M, logM, C, tw, tid, nt);
    if (MODE == 0) {
        float* o = out + (size_t)b * M * M;
        for (int i = tid; i < C * M; i += nt) {
            const int k = i / C, c = i - k * C;
            const float2 v = x[c * M + (__brev((unsigned)k) >> (32 - logM))];
            const float I = (v.x * v.x + v.y * v.y) * norm;
            const size_t gi = (size_t)k * M + m0 + c;
            o[gi] = accumulate ? o[gi] + I : I;
        }
    } else {
        for (int r = tid; r < P; r += nt) {
            float s = 0.0f;
            for (int kk = 0; kk < beta; ++kk) {
                const int kr = __brev((unsigned)(k0 + r * beta + kk)) >> (32 - logM);
                for (int c = 0; c < beta; ++c) {
                    const float2 v = x[c * M + kr];
                    s += (v.x * v.x + v.y * v.y) * norm;
                }
            }
            out[((size_t)b * P + r) * P + g] = s;
        }
    }
}

cudaError_t launch_sh_big_generic(ao_geometry* g, const WfsH& w, const float* phase, bool api_layout,
                          long long step_stride, int n_steps, float2* scratch, float* images,
                          cudaStream_t st)
{
    const int n_sel = (int)w.grp.src.size(), nsa = w.n_sub * w.n_sub;
    if (n_sel == 0 || n_steps <= 0) return cudaSuccess;
    cudaError_t e;
    const size_t smem_r = sizeof(float2) * w.M, smem_c = sizeof(float2) * (size_t)w.beta * w.M;
    e = cudaFuncSetAttribute(k_big_rows_generic, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_r);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(k_big_cols_generic<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_c);
    if (e != cudaSuccess) return e;
    const float norm = (float)(1.0 / ((double)w.M * w.M * (double)w.n * w.n));
    const int k0 = (w.M - w.beta * w.P) / 2;
    // one step at a time: the scratch holds one step of this WFS
    for (int k = 0; k < n_steps; ++k) {
        const unsigned batch = (unsigned)(n_sel * nsa);
        k_big_rows_generic<<<dim3(w.n, batch), 256, smem_r, st>>>(
            phase + (size_t)k * step_stride, step_stride, api_layout ? w.grp.d_off_api : w.grp.d_off_stage,
            n_sel, w.d_amp, w.d_valid, w.n_sub, w.n, w.M, w.logM, w.d_tw, w.d_pre, scratch);
        g->launches++;
        if ((e = cudaGetLastError()) != cudaSuccess) return e;
        k_big_cols_generic<1><<<dim3(w.P, batch), 256, smem_c, st>>>(
            scratch, w.d_valid, nsa, w.n, w.M, w.logM, w.beta, w.d_tw, norm, w.beta, w.P, k0, 0,
            images + (size_t)k * batch * w.P * w.P);
        g->launches++;
        if ((e = cudaGetLastError()) != cudaSuccess) return e;
    }
    return cudaSuccess;
}

}  // namespace ao
