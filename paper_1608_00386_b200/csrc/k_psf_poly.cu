// k_psf_poly.cu -- polychromatic science PSF (ao_psf_poly; section 2.8 "more wavelengths, considering a
// bandwidth"; DESIGN.md section 3 reading O8).
//
// Wavelength j sees the phase scaled by s = lambda_s / lambda_j and, on detector pixels of fixed angular size
// lambda_s / (M d_p), a diffraction pattern 1/s times wider: its field is the SCALED centred DFT
//     Et[k][m] = sum_ab E[a][b] exp(-2 pi i s ((k - M/2) a + (m - M/2) b) / M),   E = A exp(i s phi),
// which is not an FFT.  Each 1-D scaled DFT is evaluated as a chirp-z transform (Bluestein): with kappa = k' - M/2,
//     kappa b = (kappa^2 + b^2 - (kappa - b)^2) / 2
//     X(k') = cout[k'] * sum_b (x[b] cin[b]) h[k' - b],  cin[b] = exp(-i pi s b^2 / M),
//                                                        h[u] = exp(+i pi s (u - M/2)^2 / M),  cout[k'] = exp(-i pi s kappa^2 / M),
// a linear convolution of N inputs with M + N - 1 taps, done as a circular one of length L = 2^LOGL >= M + N - 1 through
// the register-resident Stockham FFT of fft_big.cuh:  z = IFFT_L(FFT_L(x cin) Hf),  Hf = FFT_L(h) / L (FP64, host).
// The inverse transform is the forward one on conjugates.  Tables are built in FP64 by ao_set_psf_band.
//
// Pass 1 (k_czt_rows): one CTA per pupil row: E on the fly, chirp-z along b, M outputs to the scratch T[a][m'].
// Pass 2 (k_czt_cols): one CTA per pair of columns: chirp-z along a, |.|^2 (the output chirp has unit modulus),
//   psf += w_j s_j^2 |.|^2 / (M^2 sum A^2).
#include <algorithm>

#include "fft_big.cuh"

namespace ao {

struct CztArgs {
    const float* phase; long long step_stride; const long long* off; int n_dir;   // phase of (step k, direction d)
    const float* amp; int Np, M;
    const float2* tw;          // exp(-2 pi i k / L), k < L
    const float2* cin;         // [Np]
    const float2* Hf;          // [L]
    const float2* cout;        // [M]
    float s;                   // lambda_s / lambda_j of this launch (all directions share their wavelength ratio table)
    float2* T;                 // scratch [n_dir * ks][Np][M]
    float weight;              // w_j s_j^2 / (M^2 sum A^2)
    int accumulate;
    float* psf;                // [n_dir][M][M]
    int ks;
};

__device__ __forceinline__ float2 cconj(const float2 a) { return make_float2(a.x, -a.y); }

template <int LOGL>
__global__ void __launch_bounds__((1 << LOGL) / 16)
k_czt_rows(const CztArgs A)
{
    using K = BigCfg<LOGL>;
    extern __shared__ float4 smem_raw[];
    float2* sm = reinterpret_cast<float2*>(smem_raw);
    float2* sm2 = sm + K::PADM;
    const int tb = threadIdx.x, a = blockIdx.x;
    const long long b = blockIdx.y;                                    // k * n_dir + d
    const int d = (int)(b % A.n_dir);
    const long long k = b / A.n_dir;
    const float* ph = A.phase + (size_t)k * A.step_stride + A.off[d] + (size_t)a * A.Np;
    const float* am = A.amp + (size_t)a * A.Np;
    auto sidx = [](int i) { return i + (i >> 4); };
    big_fft<LOGL>(tb, sm, 1, 0, A.tw,
        [&](int i) {
            float2 v = make_float2(0.0f, 0.0f);
            if (i < A.Np) {
                const float Am = __ldg(am + i);
                float sn, cs;
                sincos_reduced(A.s * __ldg(ph + i), &sn, &cs);
                v = cmulf(make_float2(Am * cs, Am * sn), __ldg(A.cin + i));
            }
            return v;
        },
        [&](int i, const float2 x, int) { sm2[sidx(i)] = cconj(cmulf(x, __ldg(A.Hf + i))); });
    __syncthreads();
    float2* out = A.T + ((size_t)b * A.Np + a) * A.M;
    big_fft<LOGL>(tb, sm, 1, 0, A.tw,
        [&](int i) { return sm2[sidx(i)]; },
        [&](int i, const float2 x, int) { if (i < A.M) out[i] = cmulf(cconj(x), __ldg(A.cout + i)); });
}

template <int LOGL>
__global__ void __launch_bounds__((1 << LOGL) / 8)
k_czt_cols(const CztArgs A)
{
    using K = BigCfg<LOGL>;
    constexpr int C = 2;
    extern __shared__ float4 smem_raw[];
    float2* sm = reinterpret_cast<float2*>(smem_raw);
    float2* sm2 = sm + C * K::PADM;
    const int tid = threadIdx.x, tb = tid / C, c = tid - tb * C;
    const int m = blockIdx.x * C + c;
    const int d = blockIdx.y;
    float* o = A.psf + (size_t)d * A.M * A.M + m;
    auto sidx = [&](int i) { return (i + (i >> 4)) * C + c; };
    for (int k = 0; k < A.ks; ++k) {
        const float2* Tb = A.T + ((size_t)(k * A.n_dir + d) * A.Np) * A.M + m;
        big_fft<LOGL>(tb, sm, C, c, A.tw,
            [&](int i) { return i < A.Np ? cmulf(ldg_stream(Tb + (size_t)i * A.M), __ldg(A.cin + i)) : make_float2(0.0f, 0.0f); },
            [&](int i, const float2 x, int) { sm2[sidx(i)] = cconj(cmulf(x, __ldg(A.Hf + i))); });
        __syncthreads();
        const bool add = A.accumulate || k > 0;
        big_fft<LOGL>(tb, sm, C, c, A.tw,
            [&](int i) { return sm2[sidx(i)]; },
            [&](int i, const float2 x, int) {
                if (i < A.M) {
                    const float I = A.weight * fmaf(x.x, x.x, x.y * x.y);
                    const size_t gi = (size_t)i * A.M;
                    o[gi] = add ? o[gi] + I : I;
                }
            });
        __syncthreads();                                               // the next step overwrites both buffers
    }
}

template <int LOGL>
static cudaError_t launch_czt_t(const CztArgs& a, cudaStream_t st, int64_t* launches)
{
    using K = BigCfg<LOGL>;
    const size_t smem_r = sizeof(float2) * 2 * (size_t)K::PADM, smem_c = 2 * smem_r;
    cudaError_t e;
    if ((e = cudaFuncSetAttribute(k_czt_rows<LOGL>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_r)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(k_czt_cols<LOGL>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_c)) != cudaSuccess) return e;
    k_czt_rows<LOGL><<<dim3(a.Np, a.n_dir * a.ks), K::T, smem_r, st>>>(a);
    ++*launches;
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    k_czt_cols<LOGL><<<dim3(a.M / 2, a.n_dir), K::T * 2, smem_c, st>>>(a);
    ++*launches;
    return cudaGetLastError();
}

// One wavelength of the band, ks steps (phase of step j at phase + j * step_stride), added into psf.
cudaError_t launch_psf_poly(ao_geometry* g, const float* phase, bool api_layout, long long step_stride, int ks,
                            int j, float2* scratch, float* psf, int accumulate, cudaStream_t st)
{
    const PsfBand& B = g->band;
    const int n_dir = (int)g->sci.src.size();
    if (n_dir == 0 || ks <= 0) return cudaSuccess;
    CztArgs a;
    a.phase = phase; a.step_stride = step_stride; a.off = api_layout ? g->sci.d_off_api : g->sci.d_off_stage; a.n_dir = n_dir;
    a.amp = g->d_pupil_amp; a.Np = g->Np; a.M = g->psf_fft;
    a.tw = B.d_tw; a.cin = B.d_cin + (size_t)j * g->Np; a.Hf = B.d_Hf + (size_t)j * B.L; a.cout = B.d_cout + (size_t)j * g->psf_fft;
    a.s = (float)B.scale[j]; a.T = scratch;
    a.weight = g->sumA2 > 0 ? (float)(B.weight[j] * B.scale[j] * B.scale[j] / ((double)a.M * a.M * g->sumA2)) : 0.0f;
    a.accumulate = accumulate; a.psf = psf; a.ks = ks;
    switch (B.logL) {
        case 8: return launch_czt_t<8>(a, st, &g->launches);
        case 9: return launch_czt_t<9>(a, st, &g->launches);
        case 10: return launch_czt_t<10>(a, st, &g->launches);
        case 11: return launch_czt_t<11>(a, st, &g->launches);
        case 12: return launch_czt_t<12>(a, st, &g->launches);
        default: return cudaErrorNotSupported;
    }
}

}  // namespace ao
