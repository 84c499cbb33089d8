// k_trace.cu -- stand-alone ray-trace kernel (ao_trace_layers; reading O2).
//
// One thread per output sample; layers are looped in registers.  Screen coordinates are
// carried as (integer cell, fp32 fraction): the per-(step, source, layer) origin u0 and the
// per-sample increment du are FP64, computed once per CTA into shared memory, and
// u_j = fma(j, du, u0) is evaluated in FP64 so that the fraction keeps ~1e-12 px accuracy
// even at screen coordinates of several thousand pixels (an fp32 coordinate would have
// ulp 5e-4 px there).  The interpolation itself is fp32 in difference form
//   top = s00 + fx (s01-s00), bot = s10 + fx (s11-s10), val = top + fy (bot-top)
// and the layer sum is accumulated in FP64 before the final rounding to fp32.
//
// This is the API path that materialises phase in HBM; the WFS hot path uses the fused
// kernel in k_fused.cu and never writes phase.
#include "ao_internal.cuh"

namespace ao {

__device__ __forceinline__ int wrap_index(long long i, int S, int mask)
{
    if (mask >= 0) return (int)(i & (long long)mask);
    long long r = i % S;
    return (int)(r < 0 ? r + S : r);
}

__global__ void __launch_bounds__(256)
k_trace(const LayerP* __restrict__ layers, int n_layers, const SourceP* __restrict__ srcs,
        const int* __restrict__ sel, const long long* __restrict__ off, int n_sel,
        long long step_stride, long long step0, double dt, float* __restrict__ phase)
{
    __shared__ double s_u0[kMaxLayers], s_v0[kMaxLayers], s_du[kMaxLayers];
    const int z = blockIdx.z;
    const int k = z / n_sel, si = z - k * n_sel;
    const SourceP sp = srcs[sel[si]];
    if ((int)blockIdx.x * 32 >= sp.N || (int)blockIdx.y * 8 >= sp.N) return;   // CTA-uniform
    const int tid = threadIdx.y * 32 + threadIdx.x;
    const double t = (double)(step0 + k) * dt;
    for (int l = tid; l < n_layers; l += 256) {
        const LayerP lp = layers[l];
        const double gamma = 1.0 - lp.height * sp.inv_H;
        const double x0 = -0.5 * (double)(sp.N - 1) * sp.d;
        const double c = 0.5 * (double)(lp.S - 1);
        s_u0[l] = (gamma * x0 + lp.height * sp.thx - lp.wx * t) * lp.inv_pitch + c;
        s_v0[l] = (gamma * x0 + lp.height * sp.thy - lp.wy * t) * lp.inv_pitch + c;
        s_du[l] = (lp.height < sp.H) ? gamma * sp.d * lp.inv_pitch : -1.0;   // < 0: layer skipped
    }
    __syncthreads();
    const int j = blockIdx.x * 32 + threadIdx.x, i = blockIdx.y * 8 + threadIdx.y;
    if (j >= sp.N || i >= sp.N) return;
    double acc = 0.0;
    for (int l = 0; l < n_layers; ++l) {
        const double du = s_du[l];
        if (du < 0.0) continue;
        const float* __restrict__ scr = layers[l].screen;
        const int S = layers[l].S, mask = layers[l].mask;
        const double u = fma((double)j, du, s_u0[l]);
        const double v = fma((double)i, du, s_v0[l]);
        const double fu = floor(u), fv = floor(v);
        float fx = (float)(u - fu), fy = (float)(v - fv);
        long long ju = (long long)fu, iv = (long long)fv;
        if (fx >= 1.0f) { fx = 0.0f; ++ju; }      // fraction rounded up to 1 in fp32
        if (fy >= 1.0f) { fy = 0.0f; ++iv; }
        const int j0 = wrap_index(ju, S, mask), j1 = wrap_index(ju + 1, S, mask);
        const int i0 = wrap_index(iv, S, mask), i1 = wrap_index(iv + 1, S, mask);
        const float s00 = __ldg(scr + (size_t)i0 * S + j0), s01 = __ldg(scr + (size_t)i0 * S + j1);
        const float s10 = __ldg(scr + (size_t)i1 * S + j0), s11 = __ldg(scr + (size_t)i1 * S + j1);
        const float top = fmaf(fx, s01 - s00, s00);
        const float bot = fmaf(fx, s11 - s10, s10);
        acc += (double)fmaf(fy, bot - top, top);
    }
    const size_t o = (size_t)i * sp.N + j;
    phase[(size_t)k * step_stride + off[si] + o] = (float)(acc * sp.scale + (sp.map ? (double)sp.map[o] : 0.0));
}

cudaError_t launch_trace(ao_geometry* g, const Group& grp, bool api_layout, long long step_stride,
                         int64_t step0, int n_steps, double dt, float* phase, cudaStream_t st)
{
    const int n_sel = (int)grp.src.size();
    if (n_sel == 0 || n_steps <= 0) return cudaSuccess;
    {   // fast path: TMA-staged tiles (k_fused.cu); falls through for geometries it does not cover
        const cudaError_t e = launch_trace_tiled(g, grp, api_layout, step_stride, step0, n_steps, dt, phase, st);
        if (e != cudaErrorNotSupported) return e;
    }
    dim3 block(32, 8, 1);
    const int gx = (grp.max_N + 31) / 32, gy = (grp.max_N + 7) / 8;
    // blockIdx.z is limited to 65535: split the step range if needed
    const int max_z_steps = 65535 / n_sel;
    for (int k0 = 0; k0 < n_steps; k0 += max_z_steps) {
        const int ks = (n_steps - k0 < max_z_steps) ? n_steps - k0 : max_z_steps;
        dim3 grid(gx, gy, ks * n_sel);
        k_trace<<<grid, block, 0, st>>>(g->d_layers, (int)g->layers.size(), g->d_sources, grp.d_src,
                                        api_layout ? grp.d_off_api : grp.d_off_stage, n_sel,
                                        step_stride, (long long)step0 + k0, dt,
                                        phase + (size_t)k0 * step_stride);
        g->launches++;
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

}  // namespace ao
