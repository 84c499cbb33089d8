// k_probe.cu -- FP32 peak probe: an FMA-chain micro-kernel timed with CUDA events (ao_probe_fp32).
// bench.py prints its result beside the nominal FP32 peak (148 SMs x 128 lanes x 2 x clock) so that the
// roofline denominator of the WFS forward model is a number measured in the same run on the same clocks.
#include "ao_internal.cuh"
#include "pk_tma.cuh"

namespace ao {

// 8 independent chains per thread, ITER x 8 dependent FMAs each; packed variant: FFMA2 (two FMAs per lane).
template <bool PACKED>
__global__ void __launch_bounds__(256)
k_probe_fma(float* out, const float a, const float b, const int iters)
{
    if (PACKED) {
        u64 x[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) x[i] = pack2((float)threadIdx.x + i, (float)i);
        const u64 pa = pack2(a, a), pb = pack2(b, b);
        for (int it = 0; it < iters; ++it)
#pragma unroll
            for (int r = 0; r < 8; ++r)
#pragma unroll
                for (int i = 0; i < 8; ++i) x[i] = fma2(x[i], pa, pb);
        float s = 0.0f;
#pragma unroll
        for (int i = 0; i < 8; ++i) { const float2 f = unpack2(x[i]); s += f.x + f.y; }
        if (s == 123.456f) out[0] = s;                      // never true: keeps the chains alive
    } else {
        float x[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) x[i] = (float)threadIdx.x + i;
        for (int it = 0; it < iters; ++it)
#pragma unroll
            for (int r = 0; r < 8; ++r)
#pragma unroll
                for (int i = 0; i < 8; ++i) x[i] = fmaf(x[i], a, b);
        float s = 0.0f;
#pragma unroll
        for (int i = 0; i < 8; ++i) s += x[i];
        if (s == 123.456f) out[0] = s;
    }
}

}  // namespace ao

using namespace ao;

extern "C" int ao_probe_fp32(ao_geometry* g, int packed, double* tflops_out)
{
    if (!g || !tflops_out) { set_error("ao_probe_fp32: NULL argument"); return AO_ERR_INVALID_ARG; }
    *tflops_out = 0.0;
    float* d = g->d_pupil_amp;                                       // never written: the kernel's store is unreachable
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    cudaError_t e = cudaEventCreate(&e0);
    if (e == cudaSuccess) e = cudaEventCreate(&e1);
    const int iters = 2048, ctas = g->sm_count * 8, threads = 256;
    double best = 0.0;
    for (int rep = 0; rep < 6 && e == cudaSuccess; ++rep) {          // first repetition is the warm-up
        cudaEventRecord(e0, 0);
        if (packed) k_probe_fma<true><<<ctas, threads>>>(d, 0.999f, 0.001f, iters);
        else k_probe_fma<false><<<ctas, threads>>>(d, 0.999f, 0.001f, iters);
        g->launches++;
        cudaEventRecord(e1, 0);
        e = cudaEventSynchronize(e1);
        float ms = 0.0f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
        const double flop = 2.0 * (packed ? 2.0 : 1.0) * 64.0 * iters * (double)threads * ctas;
        if (rep > 0 && ms > 0.0f && flop / (ms * 1e-3) > best) best = flop / (ms * 1e-3);
    }
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    if (e != cudaSuccess) { set_error(std::string("ao_probe_fp32: ") + cudaGetErrorString(e)); return AO_ERR_CUDA; }
    *tflops_out = best / 1e12;
    return AO_OK;
}
