// ao_device.cuh -- small device helpers shared by the CUDA kernels (noise model O5, reductions).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "ao_internal.cuh"

namespace ao {

// Philox4x32-10 (Salmon et al., SC'11), restated for the device: ten rounds of
//   (c0,c1,c2,c3) <- (hi(M1 c2)^c1^k0, lo(M1 c2), hi(M0 c0)^c3^k1, lo(M0 c0)), key += (W0, W1).
__device__ __forceinline__ uint4 philox4x32_10(uint4 c, uint32_t k0, uint32_t k1)
{
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(M0, c.x), lo0 = M0 * c.x;
        const uint32_t hi1 = __umulhi(M1, c.z), lo1 = M1 * c.z;
        c = make_uint4(hi1 ^ c.y ^ k0, lo1, hi0 ^ c.w ^ k1, lo0);
        k0 += W0; k1 += W1;
    }
    return c;
}

// u = ((w >> 8) + 0.5) 2^-24 in fp32 (rounded in the last bit above 1/2: used for the Gaussian part only; the Poisson
// decision takes the exact FP64 value, see poisson_draw).
__device__ __forceinline__ float u24(uint32_t w) { return ((float)(w >> 8) + 0.5f) * (1.0f / 16777216.0f); }

// Poisson by inversion of the CDF on u (reading O5): the smallest k with u <= F(k; mu), searched in FP64 (exp(-mu)
// underflows fp32 for mu > 87 and the integer decision must not depend on fp32 rounding of the CDF).  mu < 64: sequential
// search from 0.  mu >= 64: the same inverse CDF searched from the mode m = floor(mu) (exp(-mu) underflows FP64 above
// mu ~ 745): p_m = exp(m ln mu - mu - lgamma(m + 1)), F(m) summed downwards from the mode, then a walk down or up.
// The term ratios mu/k and j/mu are formed with a correctly rounded reciprocal and one multiplication (the oracle divides):
// the CDF then differs from the oracle's in the last bits only, which moves a decision with probability ~1e-15 per pixel,
// far inside the 1e-5 of reading O5's protocol; FP64 DDIV was most of the sampler's cost.
static __device__ __noinline__ int poisson_inv(const double mu, const double u)
{
    if (!(mu > 0.0)) return 0;
    if (mu < 64.0) {
        int k = 0;
        double p = exp(-mu), c = p;
        while (u > c && k < 100000) {
            ++k;
            p *= mu * __drcp_rn((double)k);           // mu / k up to one rounding (the oracle divides; same inverse CDF)
            c += p;
            if (p == 0.0 && (double)k > mu) break;
        }
        return k;
    }
    const double m = floor(mu), inv_mu = __drcp_rn(mu);
    const double pm = exp(m * log(mu) - mu - lgamma(m + 1.0));
    double Fm = pm, p = pm;
    for (double j = m; j >= 1.0; j -= 1.0) {
        p *= j * inv_mu;
        const double next = Fm + p;
        if (next == Fm) break;
        Fm = next;
    }
    double k = m, c = Fm;
    p = pm;
    if (u <= c) {
        while (k > 0.0 && u <= c - p) { c -= p; p *= k * inv_mu; k -= 1.0; }
    } else {
        while (u > c && k < 2147483000.0) {
            k += 1.0;
            p *= mu * __drcp_rn(k);
            c += p;
            if (p == 0.0) break;
        }
    }
    return (int)k;
}

// Fast exact filter in front of poisson_inv.  The same inverse CDF is first evaluated in fp32: search from 0 for mu < 12;
// for mu >= 12 the mode term by Stirling's series, F(mode) by the Peizer-Pratt approximation, then the same walk.  Its CDF
// values are within ~1e-5 of the FP64 ones.  If u lies further than kPoisMargin from both CDF values that bracket
// the decision, the FP64 search would take the same decision and k is returned; otherwise (about 4 u-values in 10^4, and
// always where the pmf steps are smaller than the margin: far tails, mu > 10^6) the FP64 search decides.  The integer
// decision is therefore the FP64 one of reading O5 in every case; the FP64 transcendental functions and the long FP64
// recurrences, which were 5/6 of c2's step time, run for a few pixels per thousand.
constexpr float kPoisMargin = 1.0e-4f;
// mu < 12: a few terms from k = 0 (fp32 CDF within ~2e-6 of the FP64 one).  True if the decision *kout is certain.
__device__ __forceinline__ bool poisson_small(const float muf, const float u, int* kout)
{
    int k = 0;
    float p = expf(-muf), c = p, cprev = -1.0f;
    while (u > c && k < 128) {
        ++k;
        p *= __fdividef(muf, (float)k);
        cprev = c;
        c += p;
    }
    *kout = k;
    return k < 128 && u <= c - 0.2f * kPoisMargin && u > cprev + 0.2f * kPoisMargin;
}
// 12 <= mu < 1e6: from the mode, a walk of about one standard deviation.  True if the decision *kout is certain.
__device__ __forceinline__ bool poisson_mode(const float muf, const float u, int* kout)
{
    const float m = floorf(muf), t = __fdividef(muf - m, m), inv_mu = __fdividef(1.0f, muf), im = __fdividef(1.0f, m);
    // ln p_m = m ln(mu/m) - (mu - m) - ln sqrt(2 pi m) - 1/(12 m) + 1/(360 m^3): every term is small, fp32 keeps ~1e-6
    const float im2 = im * im;
    const float lnpm = m * (log1pf(t) - t) - 0.5f * logf(6.283185307f * m) - im * (0.0833333333f - im2 * (0.00277777778f - 0.000793650794f * im2));
    const float pm = expf(lnpm);
    // F(m) by the Peizer-Pratt normal approximation (absolute error at the mode, checked against scipy.stats.poisson.cdf:
    // < 1e-5 for mu >= 8, 1.3e-6 for mu >= 16, < 2e-7 for mu in [32, 1e6]; it only has to stay far inside kPoisMargin):
    //   z = (m + 2/3 - mu + 0.02/(m+1)) sqrt((1 + g(x)) / mu),  x = (m + 1/2)/mu,  g(x) = (1 - x^2 + 2x ln x)/(1 - x)^2,
    // with g by its series in d = x - 1 (|d| <= 1/24): g = -d/3 + d^2/6 - d^3/10 + d^4/15.
    const float d = (m + 0.5f - muf) * inv_mu;
    const float g = d * (-0.333333333f + d * (0.166666667f + d * (-0.1f + d * 0.0666666667f)));
    const float z = (m - muf + 0.666666667f + __fdividef(0.02f, m + 1.0f)) * sqrtf((1.0f + g) * inv_mu);
    const float Fm = 0.5f * erfcf(-0.707106781f * z);
    float p = pm;
    float kf = m, c = Fm;
    if (u <= c) {
        while (kf > 0.0f && u <= c - p) { c -= p; p *= kf * inv_mu; kf -= 1.0f; }
    } else {
        while (u > c && kf < 2.0e6f) { kf += 1.0f; p *= __fdividef(muf, kf); c += p; if (p == 0.0f) break; }
    }
    *kout = (int)kf;
    return u <= c - kPoisMargin && u > (c - p) + kPoisMargin;      // c = F(k), c - p = F(k - 1)
}
__device__ __forceinline__ int poisson_draw(const float I_times_photons, const uint32_t w)
{
    const double ud = ((double)(w >> 8) + 0.5) * (1.0 / 16777216.0);      // exactly the oracle's u
    const double mu = (double)I_times_photons;
    const float muf = I_times_photons, u = (float)ud;
    if (!(muf > 0.0f)) return 0;
    int k = 0;
    bool sure = false;
    if (muf < 12.0f) sure = poisson_small(muf, u, &k);
    else if (muf < 1.0e6f) sure = poisson_mode(muf, u, &k);
    return sure ? k : poisson_inv(mu, ud);
}

// Detector pixel with noise (reading O5): Poisson(mu) by inversion of the CDF plus read_noise * N(0,1) (Box-Muller).
__device__ __forceinline__ float noisy_pixel(float I, const NoiseP& nz, uint32_t px, uint32_t sa,
                                             uint32_t src, uint32_t step)
{
    const uint4 w = philox4x32_10(make_uint4(px, sa, src, step), nz.key0, nz.key1);
    const int k = poisson_draw(nz.photons * I, w.x);
    const float z = sqrtf(-2.0f * logf(u24(w.y))) * cospif(2.0f * u24(w.z));
    return fmaf(nz.read_noise, z, (float)k);
}

// The same draws for NPX pixels per lane, with the long cases of the sampler shared out over the warp.  Every lane
// draws its own dim pixels (mu < 12: a few fp32 terms); the bright ones (mode start, a walk of ~sqrt(mu) steps) and the
// undecided ones (FP64 search) of all lanes are queued in `q` (shared memory of this warp, 32 NPX float2) and handed
// out lane by lane, so the warp walks them with all lanes busy instead of once per pixel slot with the few lanes that
// hold a bright pixel (c2: 3 to 7 of 32, and four unrolled copies of the sampler overflowed the instruction cache).
// v[s] = noisy_pixel(v[s], ..., px[s], ...) for lanes with `on`; all 32 lanes must call it.
template <int NPX>
__device__ __forceinline__ void noisy_pixels_warp(float (&v)[NPX], const uint32_t (&px)[NPX], const bool on, const NoiseP& nz,
                                                  const uint32_t sa, const uint32_t src, const uint32_t step, float2* q)
{
    const unsigned lane = threadIdx.x & 31u, lt = (1u << lane) - 1u;
    float z[NPX];
    int k[NPX], slot[NPX];
    int base = 0;
#pragma unroll
    for (int s = 0; s < NPX; ++s) {
        const uint4 w = philox4x32_10(make_uint4(px[s], sa, src, step), nz.key0, nz.key1);
        z[s] = sqrtf(-2.0f * logf(u24(w.y))) * cospif(2.0f * u24(w.z));
        const float muf = nz.photons * v[s];
        k[s] = 0;
        bool pend = on && muf > 0.0f;
        if (pend && muf < 12.0f) {
            const float u = (float)(((double)(w.x >> 8) + 0.5) * (1.0 / 16777216.0));
            pend = !poisson_small(muf, u, &k[s]);
        }
        const unsigned m = __ballot_sync(0xffffffffu, pend);
        slot[s] = pend ? base + __popc(m & lt) : -1;
        if (pend) q[slot[s]] = make_float2(muf, __uint_as_float(w.x));
        base += __popc(m);
    }
    __syncwarp();
    for (int j = (int)lane; j < base; j += 32) {
        const float2 e = q[j];
        const float muf = e.x;
        const double ud = ((double)(__float_as_uint(e.y) >> 8) + 0.5) * (1.0 / 16777216.0);
        int kk = 0;
        bool sure = false;
        if (muf >= 12.0f && muf < 1.0e6f) sure = poisson_mode(muf, (float)ud, &kk);
        if (!sure) kk = poisson_inv((double)muf, ud);
        q[j].x = __int_as_float(kk);
    }
    __syncwarp();
#pragma unroll
    for (int s = 0; s < NPX; ++s) {
        if (slot[s] >= 0) k[s] = __float_as_int(q[slot[s]].x);
        if (on) v[s] = fmaf(nz.read_noise, z[s], (float)k[s]);
    }
}

// sin and cos of a phase of up to a few hundred radians: exact two-constant reduction to r = x/(2 pi) - k in
// [-1/2, 1/2] revolutions, then the SFU (sin.approx / cos.approx on [-pi, pi]: absolute error ~4e-7, which the
// images see as a relative error of the same size; DESIGN.md section 5 "precision budget").
__device__ __forceinline__ void sincos_reduced(const float x, float* s, float* c)
{
    const float kInv2PiHi = 0.15915493667125702f, kInv2PiLo = 6.4206383266e-09f;
    const float k = rintf(x * kInv2PiHi);
    float r = fmaf(x, kInv2PiHi, -k);
    r = fmaf(x, kInv2PiLo, r);
    const float a = r * 6.283185307179586f;
    *s = __sinf(a);
    *c = __cosf(a);
}

// Reading O9: phase ramp of scatterer iz for the subaperture (p, q) of source-of-WFS si, in 0.32 fixed-point turns per
// sample: tau = gturn (c - L), c the subaperture centre on the O1 grid.  FP64 up to the fractional part.
__device__ __forceinline__ ElongRamp elong_ramp(const SodiumP& na, const int si, const int iz, const int p, const int q,
                                                const int n, const int N, const double d)
{
    const double g = na.gturn[si * na.n_z + iz];
    const double xc = (((double)(q * n) + 0.5 * (double)(n - 1)) - 0.5 * (double)(N - 1)) * d;
    const double yc = (((double)(p * n) + 0.5 * (double)(n - 1)) - 0.5 * (double)(N - 1)) * d;
    const double tx = g * (xc - na.launch[2 * si]), ty = g * (yc - na.launch[2 * si + 1]);
    ElongRamp r;
    r.fx = (uint32_t)__double2ull_rn((tx - floor(tx)) * 4294967296.0);
    r.fy = (uint32_t)__double2ull_rn((ty - floor(ty)) * 4294967296.0);
    return r;
}

// cos and sin of 2 pi t for t in 0.32 fixed-point turns (wrap-around is exact; SFU on [-pi, pi]).
__device__ __forceinline__ void sincos_turns(const uint32_t t, float* s, float* c)
{
    const float a = (float)(int32_t)t * (6.283185307179586f * 2.3283064365386963e-10f);
    *s = __sinf(a);
    *c = __cosf(a);
}

// A phase in radians as 0.32 fixed-point turns (same two-constant reduction as sincos_reduced).
__device__ __forceinline__ uint32_t phase_to_turns(const float x)
{
    const float kInv2PiHi = 0.15915493667125702f, kInv2PiLo = 6.4206383266e-09f;
    const float k = rintf(x * kInv2PiHi);
    float r = fmaf(x, kInv2PiHi, -k);
    r = fmaf(x, kInv2PiLo, r);                                  // [-1/2, 1/2] turns
    return (uint32_t)__float2ll_rn(r * 4294967296.0f);
}

__device__ __forceinline__ float warp_sum(float v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

}  // namespace ao
