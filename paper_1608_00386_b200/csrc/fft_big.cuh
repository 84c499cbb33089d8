// fft_big.cuh -- register-resident Stockham FFT of 64 .. 4096 points shared by the two-pass large transforms
// (k_fft_big.cu: science PSF and big-FFT sensors) and the chirp-z passes of the polychromatic PSF (k_psf_poly.cu).
// A thread holds 16 complex points, a transform of M = 2^LOGM points is T = M/16 threads and two or three
// radix-16/16/(M/256) passes; points change hands between passes through shared memory padded by one slot every 16.
#pragma once
#include "ao_device.cuh"
#include "fft_reg.cuh"

namespace ao {

template <int LOGM>
struct BigCfg {
    static constexpr int M = 1 << LOGM, T = M / 16;
    static constexpr int R1 = LOGM <= 8 ? M / 16 : 16;     // radix of the second pass
    static constexpr int R2 = LOGM <= 8 ? 1 : M / 256;     // radix of the third pass (1 = no third pass)
    static constexpr int PADM = M + M / 16;                // padded transform length in shared memory
    static_assert(LOGM >= 6 && LOGM <= 12, "big FFT sizes are 64 .. 4096");
};

__device__ __forceinline__ float2 cmulf(const float2 a, const float2 b)
{
    return make_float2(fmaf(a.x, b.x, -a.y * b.y), fmaf(a.x, b.y, a.y * b.x));
}

// Streaming load of the pass-1 intermediate: read once, strided by a whole row; kept out of L1 so that the twiddle table
// (read by every butterfly of the later passes through L1) stays there.
__device__ __forceinline__ float2 ldg_stream(const float2* p)
{
    float2 v;
    asm volatile("ld.global.nc.L1::no_allocate.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "l"(p));
    return v;
}

// Stockham pass, load half: butterfly b = tb + q T (q < 16/R) reads points b + k M/R, k < R.
template <int LOGM, int R, typename Load>
__device__ __forceinline__ void pass_load(const int tb, float2 (&v)[16], Load&& ld)
{
    constexpr int M = 1 << LOGM, T = M / 16, Q = 16 / R, STR = M / R;
#pragma unroll
    for (int q = 0; q < Q; ++q)
#pragma unroll
        for (int k = 0; k < R; ++k) v[q * R + k] = ld(tb + q * T + k * STR);
}

// Stockham pass, compute half: twiddle exp(-2 pi i (b mod NS) k / (NS R)), R-point DFT, and hand point k of
// butterfly b to st(index (b / NS) NS R + b mod NS + k NS, value, register slot).
template <int LOGM, int R, int NS, typename Store>
__device__ __forceinline__ void pass_compute(const int tb, float2 (&v)[16], const float2* __restrict__ tw, Store&& st)
{
    constexpr int M = 1 << LOGM, T = M / 16, Q = 16 / R;
#pragma unroll
    for (int q = 0; q < Q; ++q) {
        const int b = tb + q * T;
        float2 x[R];
#pragma unroll
        for (int k = 0; k < R; ++k) x[k] = v[q * R + k];
        if constexpr (NS > 1) {
            const int t0 = (b & (NS - 1)) * (M / (NS * R));
#pragma unroll
            for (int k = 1; k < R; ++k) x[k] = cmulf(x[k], __ldg(tw + t0 * k));
        }
        fft_full_pk<R>(x);
        const int o = (b / NS) * (NS * R) + (b & (NS - 1));
#pragma unroll
        for (int k = 0; k < R; ++k) st(o + k * NS, x[bitrev_c(k, R)], q * R + k);
    }
}

// One M-point forward FFT per T threads (tb = index of the thread inside its transform).  Points live in
// shared memory at sm[(i + i/16) cs + coff].  first(i) supplies input point i, last(i, value, slot) receives
// output point i (natural order; slot < 16 is a compile-time register index).  Every thread of the CTA must
// call it (it contains __syncthreads()).
template <int LOGM, typename First, typename Last>
__device__ __forceinline__ void big_fft(const int tb, float2* sm, const int cs, const int coff,
                                        const float2* __restrict__ tw, First&& first, Last&& last)
{
    using K = BigCfg<LOGM>;
    float2 v[16];
    auto sidx = [&](int i) { return (i + (i >> 4)) * cs + coff; };
    auto to_smem = [&](int i, const float2 x, int) { sm[sidx(i)] = x; };
    auto from_smem = [&](int i) { return sm[sidx(i)]; };
    pass_load<LOGM, 16>(tb, v, first);
    pass_compute<LOGM, 16, 1>(tb, v, tw, to_smem);
    __syncthreads();
    pass_load<LOGM, K::R1>(tb, v, from_smem);
    if constexpr (K::R2 == 1) {
        pass_compute<LOGM, K::R1, 16>(tb, v, tw, last);
    } else {
        __syncthreads();
        pass_compute<LOGM, K::R1, 16>(tb, v, tw, to_smem);
        __syncthreads();
        pass_load<LOGM, K::R2>(tb, v, from_smem);
        pass_compute<LOGM, K::R2, 256>(tb, v, tw, last);
    }
}

}  // namespace ao
