// k_sh_small.cu -- Shack-Hartmann image formation for FFT sizes M <= 64 from a phase buffer
// (ao_sh_images with phase_dev != NULL; readings O3, O4, O5, O6), the
// stand-alone centroid kernel (ao_centroids) and the stand-alone noise kernel.
//
// k_sh_generic: one CTA per (subaperture, source, step); works for ANY even M <= 64 (e.g. the
// M = 24 of workload c1) by evaluating the half-pixel-centred DFT as a direct separable sum
// with a shared-memory twiddle table W[q] = exp(-i pi q/M), q mod 2M:
//   R[a][m]  = sum_b E[a][b] W[((2m-M+1) b) mod 2M]          (rows,    n x M outputs)
//   E~[k][m] = sum_a R[a][m] W[((2k-M+1) a) mod 2M]          (columns, only the detector window)
// followed by |.|^2, beta x beta binning, optional noise and the centre of gravity, all inside
// the CTA.  The fused trace+SH kernel (k_fused.cu) is the hot path for M in {16,32,64}.
#include "ao_device.cuh"

namespace ao {

__global__ void __launch_bounds__(256)
k_sh_generic(const float* __restrict__ phase, long long step_stride, const long long* __restrict__ off,
             const int* __restrict__ sel, int n_sel, const float* __restrict__ amp,
             const uint8_t* __restrict__ valid, const float2* __restrict__ w2m, int n_sub, int n, int M,
             int beta, int P, float norm, NoiseP nz, long long step0, const SodiumP na, const double d_grid,
             float* __restrict__ images, float* __restrict__ slopes)
{
    extern __shared__ float4 smem_raw[];
    const int sa = blockIdx.x, si = blockIdx.y, k = blockIdx.z;
    const int nsa = n_sub * n_sub, tid = threadIdx.x, nt = blockDim.x;
    const int PP = P * P, W = beta * P, k0 = (M - W) / 2;
    const size_t set = (size_t)k * n_sel + si;
    float* img = images ? images + (set * nsa + sa) * PP : nullptr;
    float* sx = slopes ? slopes + (set * 2 + 0) * nsa + sa : nullptr;
    float* sy = slopes ? slopes + (set * 2 + 1) * nsa + sa : nullptr;
    if (!valid[sa]) {                                  // invalid subaperture: zeros
        if (img) for (int i = tid; i < PP; i += nt) img[i] = 0.0f;
        if (sx && tid == 0) { *sx = 0.0f; *sy = 0.0f; }
        return;
    }
    float2* Wt = reinterpret_cast<float2*>(smem_raw);          // [2M]
    float2* E = Wt + 2 * M;                                     // [n][n]
    float2* R = E + n * n;                                      // [n][W]   (window columns only)
    float* I = reinterpret_cast<float*>(R + n * W);             // [W][W]
    float* pix = I + W * W;                                     // [P][P]
    float2* E0 = reinterpret_cast<float2*>(pix + PP);           // [n][n]  (amplitude, phase in turns): extended beacons only
    const int p = sa / n_sub, q = sa - p * n_sub, N = n_sub * n;
    const float* ph = phase + (size_t)k * step_stride + off[si];
    for (int i = tid; i < 2 * M; i += nt) Wt[i] = w2m[i];
    const int n_z = na.n_z;                                     // 0: point beacon (one pass, no ramp)
    for (int i = tid; i < n * n; i += nt) {
        const int a = i / n, b = i - a * n;
        const size_t gidx = (size_t)(p * n + a) * N + q * n + b;
        const float A = amp[gidx];
        if (n_z > 0) {
            E0[i] = make_float2(A, __uint_as_float(phase_to_turns(ph[gidx])));
        } else {
            float s, c;
            sincos_reduced(ph[gidx], &s, &c);
            E[i] = make_float2(A * c, A * s);
        }
    }
    const float* rho = n_z > 0 ? na.rho + (size_t)((step0 + k) % na.n_t) * n_z : nullptr;
    const int twoM = 2 * M;
    for (int iz = 0; iz < (n_z > 0 ? n_z : 1); ++iz) {
        float wz = 1.0f;
        if (n_z > 0) {                                          // E = A exp(i (phi + ramp of scatterer iz)) (reading O9)
            __syncthreads();                                    // E0 written / previous scatterer's E consumed
            const ElongRamp rp = elong_ramp(na, si, iz, p, q, n, N, d_grid);
            wz = rho[iz];
            for (int i = tid; i < n * n; i += nt) {
                const int a = i / n, b = i - a * n;
                const float2 e0 = E0[i];
                float s, c;
                sincos_turns(__float_as_uint(e0.y) + (uint32_t)a * rp.fy + (uint32_t)b * rp.fx, &s, &c);
                E[i] = make_float2(e0.x * c, e0.x * s);
            }
        }
        __syncthreads();
        for (int i = tid; i < n * W; i += nt) {                 // rows
            const int a = i / W, mw = i - a * W, m = k0 + mw;
            int qs = (2 * m - M + 1) % twoM; if (qs < 0) qs += twoM;
            int qi = 0;
            float sr = 0.0f, sim = 0.0f;
            for (int b = 0; b < n; ++b) {
                const float2 x = E[a * n + b], w = Wt[qi];
                sr = fmaf(x.x, w.x, fmaf(-x.y, w.y, sr));
                sim = fmaf(x.x, w.y, fmaf(x.y, w.x, sim));
                qi += qs; if (qi >= twoM) qi -= twoM;
            }
            R[i] = make_float2(sr, sim);
        }
        __syncthreads();
        for (int i = tid; i < W * W; i += nt) {                 // columns + intensity
            const int kw = i / W, mw = i - kw * W, kk = k0 + kw;
            int qs = (2 * kk - M + 1) % twoM; if (qs < 0) qs += twoM;
            int qi = 0;
            float sr = 0.0f, sim = 0.0f;
            for (int a = 0; a < n; ++a) {
                const float2 x = R[a * W + mw], w = Wt[qi];
                sr = fmaf(x.x, w.x, fmaf(-x.y, w.y, sr));
                sim = fmaf(x.x, w.y, fmaf(x.y, w.x, sim));
                qi += qs; if (qi >= twoM) qi -= twoM;
            }
            const float v = (sr * sr + sim * sim) * norm;
            I[i] = n_z > 0 ? fmaf(wz, v, iz ? I[i] : 0.0f) : v;
        }
    }
    __syncthreads();
    for (int i = tid; i < PP; i += nt) {                        // binning (+ noise)
        const int r = i / P, c = i - r * P;
        float s = 0.0f;
        for (int y = 0; y < beta; ++y)
            for (int x = 0; x < beta; ++x) s += I[(r * beta + y) * W + c * beta + x];
        if (nz.on) s = noisy_pixel(s, nz, (uint32_t)i, (uint32_t)sa, (uint32_t)sel[si], (uint32_t)(step0 + k));
        pix[i] = s;
        if (img) img[i] = s;
    }
    __syncthreads();
    if (sx && tid < 32) {                                       // centre of gravity
        const float h = 0.5f * (float)(P - 1);
        float s = 0.0f, mx = 0.0f, my = 0.0f;
        for (int i = tid; i < PP; i += 32) {
            const int r = i / P, c = i - r * P;
            const float v = pix[i];
            s += v; mx = fmaf((float)c - h, v, mx); my = fmaf((float)r - h, v, my);
        }
        s = warp_sum(s); mx = warp_sum(mx); my = warp_sum(my);
        if (tid == 0) {
            const bool ok = fabsf(s) >= 1e-12f;
            *sx = ok ? mx / s : 0.0f;
            *sy = ok ? my / s : 0.0f;
        }
    }
}

size_t sh_generic_smem(int n, int M, int beta, int P)
{
    const size_t W = (size_t)beta * P;
    return sizeof(float2) * (2 * M + 2 * (size_t)n * n + n * W) + sizeof(float) * (W * W + (size_t)P * P) + 16;
}

cudaError_t launch_sh_small(ao_geometry* g, const WfsH& w, const float* phase, bool api_layout,
                            long long step_stride, int64_t step0, int n_steps, const NoiseP& noise,
                            float* images, float* slopes, cudaStream_t st)
{
    const int n_sel = (int)w.grp.src.size();
    if (n_sel == 0 || n_steps <= 0) return cudaSuccess;
    const size_t smem = sh_generic_smem(w.n, w.M, w.beta, w.P);
    cudaError_t e = cudaFuncSetAttribute(k_sh_generic, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const float norm = (float)(1.0 / ((double)w.M * w.M * (double)w.n * w.n));
    const int nsa = w.n_sub * w.n_sub;
    for (int k0 = 0; k0 < n_steps; k0 += 65535) {
        const int ks = n_steps - k0 < 65535 ? n_steps - k0 : 65535;
        dim3 grid(nsa, n_sel, ks);
        const size_t set0 = (size_t)k0 * n_sel;
        k_sh_generic<<<grid, 256, smem, st>>>(
            phase + (size_t)k0 * step_stride, step_stride, api_layout ? w.grp.d_off_api : w.grp.d_off_stage,
            w.grp.d_src, n_sel, w.d_amp, w.d_valid, w.d_w2m, w.n_sub, w.n, w.M, w.beta, w.P, norm, noise,
            (long long)step0 + k0, w.na, g->sources[w.grp.src[0]].d, images ? images + set0 * nsa * w.P * w.P : nullptr,
            slopes ? slopes + set0 * 2 * nsa : nullptr);
        g->launches++;
        e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

// ------------------------------------------------------------------------------------------
// Stand-alone centre of gravity (ao_centroids): one warp per image.
__global__ void __launch_bounds__(256)
k_centroid(const float* __restrict__ images, const uint8_t* __restrict__ valid, int nsa, int P,
           long long n_img, float* __restrict__ slopes)
{
    const long long img = (long long)blockIdx.x * 8 + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (img >= n_img) return;
    const long long set = img / nsa;
    const int sa = (int)(img - set * nsa);
    const float* pimg = images + (size_t)img * P * P;
    const float h = 0.5f * (float)(P - 1);
    float s = 0.0f, mx = 0.0f, my = 0.0f;
    for (int i = lane; i < P * P; i += 32) {
        const int r = i / P, c = i - r * P;
        const float v = pimg[i];
        s += v; mx = fmaf((float)c - h, v, mx); my = fmaf((float)r - h, v, my);
    }
    s = warp_sum(s); mx = warp_sum(mx); my = warp_sum(my);
    if (lane == 0) {
        const bool ok = valid[sa] && fabsf(s) >= 1e-12f;
        slopes[(size_t)(set * 2 + 0) * nsa + sa] = ok ? mx / s : 0.0f;
        slopes[(size_t)(set * 2 + 1) * nsa + sa] = ok ? my / s : 0.0f;
    }
}

// Large detectors (the 128 x 128 images of the big-FFT sensors): one CTA per image, row-wise partial sums.
__global__ void __launch_bounds__(256)
k_centroid_big(const float* __restrict__ images, const uint8_t* __restrict__ valid, int nsa, int P,
               float* __restrict__ slopes)
{
    __shared__ float red[3][8];
    const long long img = blockIdx.x;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const long long set = img / nsa;
    const int sa = (int)(img - set * nsa);
    const float* pimg = images + (size_t)img * P * P;
    const float h = 0.5f * (float)(P - 1);
    float s = 0.0f, mx = 0.0f, my = 0.0f;
    for (int r = warp; r < P; r += 8) {                       // a warp per detector row
        float rs = 0.0f;
        for (int c = lane; c < P; c += 32) {
            const float v = pimg[(size_t)r * P + c];
            rs += v; mx = fmaf((float)c - h, v, mx);
        }
        s += rs; my = fmaf((float)r - h, rs, my);
    }
    s = warp_sum(s); mx = warp_sum(mx); my = warp_sum(my);
    if (lane == 0) { red[0][warp] = s; red[1][warp] = mx; red[2][warp] = my; }
    __syncthreads();
    if (threadIdx.x == 0) {
        s = 0.0f; mx = 0.0f; my = 0.0f;
        for (int w = 0; w < 8; ++w) { s += red[0][w]; mx += red[1][w]; my += red[2][w]; }
        const bool ok = valid[sa] && fabsf(s) >= 1e-12f;
        slopes[(size_t)(set * 2 + 0) * nsa + sa] = ok ? mx / s : 0.0f;
        slopes[(size_t)(set * 2 + 1) * nsa + sa] = ok ? my / s : 0.0f;
    }
}

cudaError_t launch_centroids(ao_geometry* g, const WfsH& w, const float* images, int n_sets,
                             float* slopes, cudaStream_t st)
{
    const int nsa = w.n_sub * w.n_sub;
    const long long n_img = (long long)n_sets * nsa;
    if (n_img <= 0) return cudaSuccess;
    if (w.P >= 64 && n_img <= 0x7fffffffLL) {
        k_centroid_big<<<(unsigned)n_img, 256, 0, st>>>(images, w.d_valid, nsa, w.P, slopes);
        g->launches++;
        return cudaGetLastError();
    }
    const long long blocks = (n_img + 7) / 8;
    k_centroid<<<(unsigned)blocks, 256, 0, st>>>(images, w.d_valid, nsa, w.P, n_img, slopes);
    g->launches++;
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------
// ao_modes_to_map: map[i] = sign * sum_m coeffs[m] modes[m][i] (PAPER.md:82 residual phase, :74 calibration pushes).
// HBM-bound: every mode array is read once, coalesced; the coefficients are warp-uniform loads.
__global__ void __launch_bounds__(256)
k_modes_to_map(const float* __restrict__ modes, int n_modes, long long n_elems, const float* __restrict__ coeffs,
               float sign, float* __restrict__ map)
{
    const long long i = (long long)blockIdx.x * 256 + threadIdx.x;
    if (i >= n_elems) return;
    float acc = 0.0f;
    for (int m = 0; m < n_modes; ++m) acc = fmaf(__ldg(coeffs + m), modes[(size_t)m * n_elems + i], acc);
    map[i] = sign * acc;
}

cudaError_t launch_modes_to_map(ao_geometry* g, const float* modes, int n_modes, long long n_elems, const float* coeffs,
                                float sign, float* map, cudaStream_t st)
{
    if (n_elems <= 0) return cudaSuccess;
    k_modes_to_map<<<(unsigned)((n_elems + 255) / 256), 256, 0, st>>>(modes, n_modes, n_elems, coeffs, sign, map);
    g->launches++;
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------
// ao_strehl: peak pixel [M/2][M/2] of every long-exposure PSF over the diffraction-limited peak.
__global__ void k_strehl(const float* __restrict__ psf, int n_dir, int M, float inv_norm, float* __restrict__ strehl)
{
    const int d = blockIdx.x * blockDim.x + threadIdx.x;
    if (d < n_dir) strehl[d] = psf[((size_t)d * M + M / 2) * M + M / 2] * inv_norm;
}

cudaError_t launch_strehl(ao_geometry* g, const float* psf, int n_dir, int M, float inv_norm, float* strehl, cudaStream_t st)
{
    k_strehl<<<(n_dir + 63) / 64, 64, 0, st>>>(psf, n_dir, M, inv_norm, strehl);
    g->launches++;
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------
// ao_strehl_marechal: exp(-amplitude-weighted phase variance) per (step, science direction); one CTA each, FP64 sums
// of w, w phi, w phi^2 (phase is tens of radians in open loop: the difference of squares needs the headroom).
__global__ void __launch_bounds__(256)
k_marechal(const float* __restrict__ phase, long long step_stride, const long long* __restrict__ off, int n_dir,
           const float* __restrict__ amp, int N, float* __restrict__ strehl)
{
    __shared__ double red[3][8];
    const int d = blockIdx.x % n_dir, k = blockIdx.x / n_dir;
    const float* ph = phase + (size_t)k * step_stride + off[d];
    double sw = 0.0, s1 = 0.0, s2 = 0.0;
    for (size_t i = threadIdx.x; i < (size_t)N * N; i += 256) {
        const double w = (double)amp[i], p = (double)ph[i];
        sw += w; s1 += w * p; s2 += w * p * p;
    }
    for (int o = 16; o > 0; o >>= 1) {
        sw += __shfl_xor_sync(0xffffffffu, sw, o); s1 += __shfl_xor_sync(0xffffffffu, s1, o); s2 += __shfl_xor_sync(0xffffffffu, s2, o);
    }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (lane == 0) { red[0][warp] = sw; red[1][warp] = s1; red[2][warp] = s2; }
    __syncthreads();
    if (threadIdx.x == 0) {
        sw = s1 = s2 = 0.0;
        for (int w = 0; w < 8; ++w) { sw += red[0][w]; s1 += red[1][w]; s2 += red[2][w]; }
        double var = 0.0;
        if (sw > 0.0) { const double mean = s1 / sw; var = s2 / sw - mean * mean; if (var < 0.0) var = 0.0; }
        strehl[blockIdx.x] = (float)exp(-var);
    }
}

cudaError_t launch_marechal(ao_geometry* g, const float* phase, long long step_stride, int n_steps, float* strehl,
                            cudaStream_t st)
{
    const int n_dir = (int)g->sci.src.size();
    if (n_dir == 0 || n_steps <= 0) return cudaSuccess;
    k_marechal<<<(unsigned)(n_dir * n_steps), 256, 0, st>>>(phase, step_stride, g->sci.d_off_api, n_dir, g->d_pupil_amp,
                                                            g->Np, strehl);
    g->launches++;
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------
// Stand-alone detector noise, in place on [n_steps][n_sel][nsa][P][P] normalised images.
__global__ void __launch_bounds__(256)
k_noise(float* __restrict__ images, const uint8_t* __restrict__ valid, const int* __restrict__ sel,
        int n_sel, int nsa, int PP, long long total, long long step0, NoiseP nz)
{
    const long long i = (long long)blockIdx.x * 256 + threadIdx.x;
    if (i >= total) return;
    const int px = (int)(i % PP);
    const long long t = i / PP;
    const int sa = (int)(t % nsa);
    const long long set = t / nsa;
    const int si = (int)(set % n_sel);
    const long long k = set / n_sel;
    if (!valid[sa]) { images[i] = 0.0f; return; }
    images[i] = noisy_pixel(images[i], nz, (uint32_t)px, (uint32_t)sa, (uint32_t)sel[si], (uint32_t)(step0 + k));
}

cudaError_t launch_noise(ao_geometry* g, const WfsH& w, float* images, int64_t step0, int n_steps,
                         const NoiseP& noise, cudaStream_t st)
{
    const int n_sel = (int)w.grp.src.size(), nsa = w.n_sub * w.n_sub, PP = w.P * w.P;
    const long long total = (long long)n_steps * n_sel * nsa * PP;
    if (total <= 0) return cudaSuccess;
    k_noise<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(images, w.d_valid, w.grp.d_src, n_sel, nsa, PP,
                                                            total, (long long)step0, noise);
    g->launches++;
    return cudaGetLastError();
}

}  // namespace ao
