// k_sh_reg.cu -- Shack-Hartmann image formation from a phase buffer with in-register FFTs, for the sensor shapes
// M in {16, 24, 32, 64}, n = M/2, full detector window (beta P = M): workloads c0 (16), c1 (24: 3 x 4 x 2 Cooley-Tukey,
// fft12 of fft_reg.cuh) and c2-c4 (32) when ao_sh_images is called with a phase buffer, c1's phase_dev == NULL path
// after the tiled ray-trace, and c4 at M = 64 (one warp per subaperture, 32-point FFTs in registers).  PAPER.md:28,82; readings O3, O4, O5, O6.  Other shapes run k_sh_generic (direct DFT).
//
// A group of n threads owns one subaperture (thread b = column b): E[a] = A exp(i phi) of its column, the half-pixel
// centred M-point column DFT in registers (dft_half_padded: two n-point FFTs with compile-time twiddles), one transpose
// through padded shared memory, the row DFTs of rows b and b + n, |.|^2 summed over the beta columns of a detector
// pixel in registers, the beta rows through shared memory; then noise, image store and centre of gravity.
#include "ao_device.cuh"
#include "fft_reg.cuh"

namespace ao {

struct ShRegArgs {
    const float* phase; long long step_stride; const long long* off;
    const int* sel; int n_sel;
    const float* amp; const uint8_t* valid; int n_sub, nsa;
    float norm; NoiseP nz; long long step0;
    long long total;                  // n_steps * n_sel * nsa
    float* images; float* slopes;
};

template <int M, int BETA>
__global__ void __launch_bounds__(128)
k_sh_reg(const ShRegArgs A)
{
    constexpr int n = M / 2, P = M / BETA, XP = n + 1, GPW = 32 / n, GPC = 4 * GPW;      // groups per warp / per CTA
    constexpr int SUB_F2 = M * XP;                                                      // float2 per group: T[k][b]
    constexpr int SUB_F = M * P + P * P;                                                // floats per group: row bins, pixels
    extern __shared__ float4 smem_raw[];
    float2* xch = reinterpret_cast<float2*>(smem_raw);                                  // [GPC][SUB_F2]
    float* fbuf = reinterpret_cast<float*>(xch + GPC * SUB_F2);                         // [GPC][SUB_F]
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int gw = lane / n, b = lane - gw * n;                 // group in warp, column in subaperture
    const bool lane_on = gw < GPW;                              // n = 12: lanes 24..31 idle
    const int grp = warp * GPW + (lane_on ? gw : 0);
    const long long item = (long long)blockIdx.x * GPC + grp;  // (step k, source si, subaperture sa)
    const bool item_on = lane_on && item < A.total;
    const int sa = item_on ? (int)(item % A.nsa) : 0;
    const long long set = item_on ? item / A.nsa : 0;
    const int si = (int)(set % A.n_sel);
    const long long k = set / A.n_sel;
    const bool active = item_on && A.valid[sa] != 0;
    float2* xs = xch + grp * SUB_F2;
    float* rb = fbuf + grp * SUB_F;
    float* pix = rb + M * P;
    const int p = sa / A.n_sub, q = sa - p * A.n_sub, N = A.n_sub * n;
    if (!__any_sync(0xffffffffu, active)) {                    // no lit subaperture in this warp: zeros, no transform
        if (item_on) {
            if (A.images) for (int px = b; px < P * P; px += n) A.images[(size_t)item * (P * P) + px] = 0.0f;
            if (A.slopes && b == 0) {
                A.slopes[((size_t)set * 2 + 0) * A.nsa + sa] = 0.0f;
                A.slopes[((size_t)set * 2 + 1) * A.nsa + sa] = 0.0f;
            }
        }
        return;
    }
    {
        float2 e[n];
        const size_t base = (size_t)(p * n) * N + (size_t)q * n + b;
        const float* ph = A.phase + (size_t)k * A.step_stride + A.off[si] + base;
        const float* am = A.amp + base;
#pragma unroll
        for (int i = 0; i < n; ++i) {
            float s = 0.0f, c = 0.0f, Am = 0.0f;
            if (active) { Am = __ldg(am + (size_t)i * N); sincos_reduced(__ldg(ph + (size_t)i * N), &s, &c); }
            e[i] = make_float2(Am * c, Am * s);
        }
        dft_half_padded<M>(e, [&](auto ki, const float2 v) {
            constexpr int kk = decltype(ki)::value;
            if (lane_on) xs[kk * XP + b] = v;
        });
    }
    __syncwarp();
#pragma unroll
    for (int hh = 0; hh < 2; ++hh) {                            // rows b and b + n
        const int kr = b + hh * n;
        float2 rrow[n];
#pragma unroll
        for (int i = 0; i < n; ++i) rrow[i] = lane_on ? xs[kr * XP + i] : make_float2(0.0f, 0.0f);
        float bins[P];
#pragma unroll
        for (int i = 0; i < P; ++i) bins[i] = 0.0f;
        dft_half_padded<M>(rrow, [&](auto mi, const float2 v) {
            constexpr int m = decltype(mi)::value;
            bins[m / BETA] = fmaf(v.x, v.x, fmaf(v.y, v.y, bins[m / BETA]));
        });
        if (lane_on) {
#pragma unroll
            for (int i = 0; i < P; ++i) rb[kr * P + i] = bins[i];
        }
    }
    __syncwarp();
    float s = 0.0f, mx = 0.0f, my = 0.0f;
    const float hP = 0.5f * (float)(P - 1);
    if (item_on) {
        float* img = A.images ? A.images + (size_t)item * (P * P) : nullptr;
        for (int px = b; px < P * P; px += n) {                 // detector pixel = sum of its beta rows
            const int r = px / P, c = px - r * P;
            float v = 0.0f;
#pragma unroll
            for (int y = 0; y < BETA; ++y) v += rb[(r * BETA + y) * P + c];
            v *= A.norm;
            if (active && A.nz.on) v = noisy_pixel(v, A.nz, (uint32_t)px, (uint32_t)sa, (uint32_t)A.sel[si], (uint32_t)(A.step0 + k));
            if (!active) v = 0.0f;
            if (img) img[px] = v;
            pix[px] = v;
            s += v; mx = fmaf((float)c - hP, v, mx); my = fmaf((float)r - hP, v, my);
        }
    }
    if constexpr ((n & (n - 1)) == 0) {                          // centre of gravity: butterfly over the group's n lanes
#pragma unroll
        for (int o = n / 2; o >= 1; o >>= 1) {
            s += __shfl_xor_sync(0xffffffffu, s, o);
            mx += __shfl_xor_sync(0xffffffffu, mx, o);
            my += __shfl_xor_sync(0xffffffffu, my, o);
        }
    } else {                                                     // n = 12: the group's first lane sums the pixels in order
        __syncwarp();
        if (item_on && b == 0) {
            s = 0.0f; mx = 0.0f; my = 0.0f;
            for (int px = 0; px < P * P; ++px) {
                const int r = px / P, c = px - r * P;
                const float v = pix[px];
                s += v; mx = fmaf((float)c - hP, v, mx); my = fmaf((float)r - hP, v, my);
            }
        }
    }
    if (item_on && b == 0 && A.slopes) {
        const bool ok = active && fabsf(s) >= 1e-12f;
        A.slopes[((size_t)set * 2 + 0) * A.nsa + sa] = ok ? mx / s : 0.0f;
        A.slopes[((size_t)set * 2 + 1) * A.nsa + sa] = ok ? my / s : 0.0f;
    }
}

bool sh_reg_supported(const WfsH& w)
{
    if (w.n * 2 != w.M || w.beta * w.P != w.M || w.na.n_z > 0) return false;
    return (w.M == 16 && w.beta == 2) || (w.M == 24 && w.beta == 4) || (w.M == 32 && w.beta == 4) || (w.M == 64 && w.beta == 8);
}

cudaError_t launch_sh_reg(ao_geometry* g, const WfsH& w, const float* phase, bool api_layout, long long step_stride,
                          int64_t step0, int n_steps, const NoiseP& noise, float* images, float* slopes, cudaStream_t st)
{
    const int n_sel = (int)w.grp.src.size();
    if (n_sel == 0 || n_steps <= 0) return cudaSuccess;
    ShRegArgs a;
    a.phase = phase; a.step_stride = step_stride; a.off = api_layout ? w.grp.d_off_api : w.grp.d_off_stage;
    a.sel = w.grp.d_src; a.n_sel = n_sel; a.amp = w.d_amp; a.valid = w.d_valid; a.n_sub = w.n_sub; a.nsa = w.n_sub * w.n_sub;
    a.norm = (float)(1.0 / ((double)w.M * w.M * (double)w.n * w.n));
    a.nz = noise; a.step0 = (long long)step0; a.total = (long long)n_steps * n_sel * a.nsa;
    a.images = images; a.slopes = slopes;
    const int gpc = 4 * (32 / w.n);
    const long long blocks = (a.total + gpc - 1) / gpc;
    if (blocks > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    const int P = w.P;
    const size_t smem = (size_t)gpc * (sizeof(float2) * w.M * (w.n + 1) + sizeof(float) * (w.M * P + P * P));
    void (*kern)(const ShRegArgs) = w.M == 16 ? k_sh_reg<16, 2> : w.M == 24 ? k_sh_reg<24, 4> : w.M == 32 ? k_sh_reg<32, 4> : k_sh_reg<64, 8>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    kern<<<(unsigned)blocks, 128, smem, st>>>(a);
    g->launches++;
    return cudaGetLastError();
}

}  // namespace ao
