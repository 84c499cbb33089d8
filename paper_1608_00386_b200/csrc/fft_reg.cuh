// fft_reg.cuh -- in-register FFT building blocks with compile-time twiddles, shared by the fused
// Shack-Hartmann kernel (k_fused.cu) and the big two-pass FFT (k_fft_big.cu).
// Readings O3 / O7 of DESIGN.md section 3 (centred DFTs of the SH sensor and of the science PSF).
#pragma once
#include <cuda_runtime.h>
#include <type_traits>

#include "pk_tma.cuh"

namespace ao {

// ---- compile-time trigonometry and complex constants ----
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

// Packed-complex variant of fft_stage (fft_reg.cuh): a complex number is one f32x2 register pair, so the
// butterfly add and subtract are one FADD2 each; twiddle multiplications stay scalar.
template <int NUM, int DEN>
__device__ __forceinline__ u64 cmul_cis_pk(const u64 x)
{
    using W = Cis<NUM, DEN>;
    if constexpr (W::q == 0) return x;
    else { const float2 r = cmul_cis<NUM, DEN>(unpack2(x)); return pack2(r.x, r.y); }
}
template <int N, int HALF>
__device__ __forceinline__ void fft_stage_pk(u64 (&x)[N])
{
    static_for<0, N / 2>([&](auto bi) {
        constexpr int b = decltype(bi)::value;
        constexpr int grp = b / HALF, pos = b % HALF, i = grp * 2 * HALF + pos, j = i + HALF;
        const u64 a = x[i], c = x[j];
        x[i] = add2(a, c);
        x[j] = cmul_cis_pk<-pos, HALF>(sub2(a, c));                            // * exp(-2 pi i pos/(2 HALF))
    });
    if constexpr (HALF > 1) fft_stage_pk<N, HALF / 2>(x);
}

// fft_stage on a float2 array through the packed butterflies (R-point DFT of the big-FFT passes).
template <int N>
__device__ __forceinline__ void fft_full_pk(float2 (&x)[N])
{
    if constexpr (N > 1) {
        u64 y[N];
#pragma unroll
        for (int i = 0; i < N; ++i) y[i] = pack2(x[i].x, x[i].y);
        fft_stage_pk<N, N / 2>(y);
#pragma unroll
        for (int i = 0; i < N; ++i) x[i] = unpack2(y[i]);
    }
}

}  // namespace ao
