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

// 12-point forward DFT in registers (3 x 4 Cooley-Tukey, compile-time twiddles), natural order in and out:
// a = 4 a1 + a2, k = k1 + 3 k2:  X[k1 + 3 k2] = sum_a2 W4^(a2 k2) [ W12^(a2 k1) sum_a1 x[4 a1 + a2] W3^(a1 k1) ].
__device__ __forceinline__ void fft12(float2 (&x)[12])
{
    float2 t[3][4];
    static_for<0, 4>([&](auto a2i) {
        constexpr int a2 = decltype(a2i)::value;
        const float2 p = x[a2], q = x[4 + a2], r = x[8 + a2];
        const float2 s = make_float2(q.x + r.x, q.y + r.y), d = make_float2(q.x - r.x, q.y - r.y);
        const float2 m = make_float2(fmaf(-0.5f, s.x, p.x), fmaf(-0.5f, s.y, p.y));
        const float h = 0.86602540378443864676f;                        // sqrt(3)/2; -i d = (d.y, -d.x)
        const float2 t0 = make_float2(p.x + s.x, p.y + s.y);
        const float2 t1 = make_float2(fmaf(h, d.y, m.x), fmaf(-h, d.x, m.y));
        const float2 t2 = make_float2(fmaf(-h, d.y, m.x), fmaf(h, d.x, m.y));
        t[0][a2] = t0;
        t[1][a2] = cmul_cis<-a2, 6>(t1);                                 // W12^(a2 k1) = cis(-pi a2 k1 / 6)
        t[2][a2] = cmul_cis<-2 * a2, 6>(t2);
    });
    static_for<0, 3>([&](auto k1i) {
        constexpr int k1 = decltype(k1i)::value;
        const float2 a = t[k1][0], b = t[k1][1], c = t[k1][2], d = t[k1][3];
        const float2 ac = make_float2(a.x + c.x, a.y + c.y), amc = make_float2(a.x - c.x, a.y - c.y);
        const float2 bd = make_float2(b.x + d.x, b.y + d.y), bmd = make_float2(b.x - d.x, b.y - d.y);
        x[k1] = make_float2(ac.x + bd.x, ac.y + bd.y);
        x[k1 + 6] = make_float2(ac.x - bd.x, ac.y - bd.y);
        x[k1 + 3] = make_float2(amc.x + bmd.y, amc.y - bmd.x);           // - i (b - d)
        x[k1 + 9] = make_float2(amc.x - bmd.y, amc.y + bmd.x);           // + i (b - d)
    });
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
    if constexpr (n == 12) {                                           // M = 24 (workload c1): 12-point FFTs, 3 x 4
        float2 y[n];
        static_for<0, n>([&](auto ai) { constexpr int a = decltype(ai)::value; y[a] = cmul_cis<(M - 1) * a, M>(e[a]); });
        fft12(y);
        static_for<0, n>([&](auto ki) { constexpr int k = decltype(ki)::value; sink(std::integral_constant<int, 2 * k>{}, y[k]); });
        static_for<0, n>([&](auto ai) { constexpr int a = decltype(ai)::value; y[a] = cmul_cis<(M - 3) * a, M>(e[a]); });
        fft12(y);
        static_for<0, n>([&](auto ki) { constexpr int k = decltype(ki)::value; sink(std::integral_constant<int, 2 * k + 1>{}, y[k]); });
        return;
    }
    else {
    u64 y[n];
    static_for<0, n>([&](auto ai) { constexpr int a = decltype(ai)::value; const float2 t = cmul_cis<(M - 1) * a, M>(e[a]); y[a] = pack2(t.x, t.y); });
    fft_stage_pk<n, n / 2>(y);
    static_for<0, n>([&](auto ki) { constexpr int k = decltype(ki)::value; sink(std::integral_constant<int, 2 * k>{}, unpack2(y[bitrev_c(k, n)])); });
    static_for<0, n>([&](auto ai) { constexpr int a = decltype(ai)::value; const float2 t = cmul_cis<(M - 3) * a, M>(e[a]); y[a] = pack2(t.x, t.y); });
    fft_stage_pk<n, n / 2>(y);
    static_for<0, n>([&](auto ki) { constexpr int k = decltype(ki)::value; sink(std::integral_constant<int, 2 * k + 1>{}, unpack2(y[bitrev_c(k, n)])); });
    }
}


}  // namespace ao
