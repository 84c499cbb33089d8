// ao_api.cu -- host side of libao.so: the extern "C" entry points declared in include/ao.h.
// Validation, device tables, workspace planning and launch sequencing only; every number of
// the forward model is produced by the kernels in k_*.cu.
#include <cmath>
#include <complex>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>

#include "ao_internal.cuh"

namespace ao {

static thread_local std::string g_err = "";
void set_error(const std::string& msg) { g_err = msg; }

static int fail(int code, const std::string& msg) { set_error(msg); return code; }
static int cuda_fail(cudaError_t e, const char* what)
{
    return fail(AO_ERR_CUDA, std::string(what) + ": " + cudaGetErrorString(e));
}

#define AO_CUDA(call, what) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) return cuda_fail(e__, what); } while (0)

static bool is_pow2(int v) { return v > 0 && (v & (v - 1)) == 0; }
static int ilog2(int v) { int l = 0; while ((1 << l) < v) ++l; return l; }
static size_t align256(size_t v) { return (v + 255) & ~(size_t)255; }

template <typename T>
static cudaError_t upload(T** dptr, const T* host, size_t count)
{
    *dptr = nullptr;
    if (count == 0) return cudaSuccess;
    cudaError_t e = cudaMalloc((void**)dptr, sizeof(T) * count);
    if (e != cudaSuccess) return e;
    return cudaMemcpy(*dptr, host, sizeof(T) * count, cudaMemcpyHostToDevice);
}

static cudaError_t build_group(ao_geometry* g, Group& grp)
{
    std::vector<long long> off_api, off_stage;
    long long acc = 0;
    grp.max_N = 0;
    for (int s : grp.src) {
        const SourceP& sp = g->sources[s];
        off_api.push_back(sp.phase_off);
        off_stage.push_back(acc);
        acc += (long long)sp.N * sp.N;
        if (sp.N > grp.max_N) grp.max_N = sp.N;
    }
    grp.stage_elems = acc;
    cudaError_t e;
    if ((e = upload(&grp.d_src, grp.src.data(), grp.src.size())) != cudaSuccess) return e;
    if ((e = upload(&grp.d_off_api, off_api.data(), off_api.size())) != cudaSuccess) return e;
    return upload(&grp.d_off_stage, off_stage.data(), off_stage.size());
}

static void free_sodium(WfsH& w)
{
    cudaFree((void*)w.na.rho); cudaFree((void*)w.na.gturn); cudaFree((void*)w.na.launch);
    w.na = SodiumP();
}

static void free_band(ao_geometry* g)
{
    cudaFree(g->band.d_tw); cudaFree(g->band.d_cin); cudaFree(g->band.d_Hf); cudaFree(g->band.d_cout);
    g->band = PsfBand();
}

static void free_group(Group& grp)
{
    cudaFree(grp.d_src); cudaFree(grp.d_off_api); cudaFree(grp.d_off_stage);
    grp.d_src = nullptr; grp.d_off_api = nullptr; grp.d_off_stage = nullptr;
}

static void destroy(ao_geometry* g)
{
    if (!g) return;
    cudaFree(g->d_pupil_amp); cudaFree(g->d_layers); cudaFree(g->d_sources);
    cudaFree(g->d_psf_tw); cudaFree(g->d_psf_pre);
    free_band(g);
    for (auto& w : g->wfs) {
        cudaFree(w.d_amp); cudaFree(w.d_valid); cudaFree(w.d_w2m); cudaFree(w.d_tw); cudaFree(w.d_twf); cudaFree(w.d_pre); cudaFree(w.fused_items);
        free_sodium(w);
        cudaFree(w.d_tmaps);
        free_group(w.grp);
    }
    free_group(g->all); free_group(g->sci);
    delete g;
}

// ---- workspace planning ---------------------------------------------------------------------
struct Plan {
    size_t scratch = 0;     // FFT scratch (one step of the largest big transform batch)
    size_t fixed = 0;       // PSF staging for ao_forward_host
    size_t stage = 0;       // per step: phase staging (largest group)
    size_t bigimg = 0;      // per step: images of the largest big WFS
    size_t slopes = 0;      // per step: slopes of all WFS (ao_forward_host staging)
    size_t per_step() const { return stage + bigimg + slopes; }
};

static Plan make_plan(const ao_geometry* g)
{
    Plan p;
    size_t stage_elems = 0;
    if (g->psf_fft && !g->sci.src.empty()) {
        p.scratch = psf_scratch_bytes(g) * (size_t)psf_chunk_steps(g);
        p.fixed = align256(sizeof(float) * g->sci.src.size() * (size_t)g->psf_fft * g->psf_fft);
        stage_elems = (size_t)g->sci.stage_elems;
    }
    for (const auto& w : g->wfs) {
        const size_t n_sel = w.grp.src.size(), nsa = (size_t)w.n_sub * w.n_sub;
        if ((size_t)w.grp.stage_elems > stage_elems) stage_elems = (size_t)w.grp.stage_elems;
        p.slopes += align256(sizeof(float) * n_sel * 2 * nsa);
        if (w.big) {
            size_t s = sh_big_scratch_bytes(g, w);
            int kb = 8;                                      // up to 8 steps per launch pair within 768 MB of intermediate
            while (kb > 1 && (size_t)kb * s > ((size_t)768 << 20)) --kb;
            s *= (size_t)kb;
            if (s > p.scratch) p.scratch = s;
            const size_t im = align256(sizeof(float) * n_sel * nsa * w.P * w.P);
            if (im > p.bigimg) p.bigimg = im;
        }
    }
    p.scratch = align256(p.scratch);
    p.stage = align256(sizeof(float) * stage_elems);
    return p;
}

struct WsView {
    float2* scratch; float* psf_stage; float* stage; float* bigimg; float* slopes; int chunk;
};

static WsView ws_view(const ao_geometry* g)
{
    const Plan p = make_plan(g);
    WsView v;
    char* b = g->ws;
    v.chunk = g->ws_chunk;
    v.scratch = (float2*)b; b += p.scratch;
    v.psf_stage = (float*)b; b += p.fixed;
    v.stage = (float*)b; b += p.stage * (size_t)v.chunk;
    v.bigimg = (float*)b; b += p.bigimg * (size_t)v.chunk;
    v.slopes = (float*)b;
    return v;
}

static NoiseP make_noise(const ao_noise* nz)
{
    NoiseP p; memset(&p, 0, sizeof(p));
    if (nz) {
        p.on = 1; p.key0 = (uint32_t)nz->seed; p.key1 = (uint32_t)(nz->seed >> 32);
        p.photons = nz->photons_per_subap; p.read_noise = nz->read_noise_e;
    }
    return p;
}

// Entry check of every compute call: the handle, the device it was created on (made current for this thread
// if it is not), and errors left by earlier asynchronous work.  The error is only peeked at: errors raised by
// other libraries in the same process stay theirs to consume.
static int check_entry(const ao_geometry* g)
{
    if (!g) return fail(AO_ERR_INVALID_ARG, "NULL handle");
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess && dev != g->device) e = cudaSetDevice(g->device);
    if (e != cudaSuccess) return cuda_fail(e, "selecting the handle's device");
    e = cudaPeekAtLastError();
    if (e != cudaSuccess) return cuda_fail(e, "pending CUDA error from earlier work");
    return AO_OK;
}

// Run SH (+noise, +CoG) of WFS w for steps [step0, step0+n_steps), chunked by the workspace.
static int run_wfs(ao_geometry* g, int wi, const float* phase_dev, int64_t step0, int n_steps, double dt,
                   const ao_noise* noise, float* images, float* slopes, cudaStream_t st)
{
    WfsH& w = g->wfs[wi];
    const size_t n_sel = w.grp.src.size(), nsa = (size_t)w.n_sub * w.n_sub, PP = (size_t)w.P * w.P;
    if (n_sel == 0) return AO_OK;
    if (!phase_dev && (!w.big || w.M == 64)) {        // hot path: one fused kernel, no phase in HBM, no workspace
        if (fused_supported(g, w, dt)) {
            AO_CUDA(launch_fused(g, w, step0, n_steps, dt, make_noise(noise), images, slopes, st), "fused");
            return AO_OK;
        }
    }
    // M = 64 is grouped with the big sensors for its tables; it runs k_sh_reg (n = 32, 8 x 8 bins of the whole field),
    // k_sh_generic for an extended beacon, else the one-CTA-per-subaperture Stockham kernel k_sh_mid64
    const bool big = w.big && !(w.M <= 64 && (w.na.n_z > 0 || sh_reg_supported(w)));
    const bool need_ws = (phase_dev == nullptr) || big;
    if (need_ws && (!g->ws || g->ws_chunk < 1))
        return fail(AO_ERR_WORKSPACE, "workspace required (phase_dev == NULL or fft > 64): call ao_set_workspace");
    const NoiseP nz = make_noise(noise);
    const WsView v = need_ws ? ws_view(g) : WsView{};
    const int chunk = need_ws ? v.chunk : n_steps;
    for (int c0 = 0; c0 < n_steps; c0 += chunk) {
        const int ks = (n_steps - c0 < chunk) ? n_steps - c0 : chunk;
        const float* ph; bool api; long long stride;
        if (phase_dev) {
            ph = phase_dev + (size_t)c0 * g->phase_elems_per_step; api = true; stride = g->phase_elems_per_step;
        } else {
            AO_CUDA(launch_trace(g, w.grp, false, w.grp.stage_elems, step0 + c0, ks, dt, v.stage, st), "trace");
            ph = v.stage; api = false; stride = w.grp.stage_elems;
        }
        float* img = images ? images + (size_t)c0 * n_sel * nsa * PP : nullptr;
        float* slp = slopes ? slopes + (size_t)c0 * n_sel * 2 * nsa : nullptr;
        if (!big) {
            if (sh_reg_supported(w)) AO_CUDA(launch_sh_reg(g, w, ph, api, stride, step0 + c0, ks, nz, img, slp, st), "sh_reg");
            else AO_CUDA(launch_sh_small(g, w, ph, api, stride, step0 + c0, ks, nz, img, slp, st), "sh_small");
        } else {
            float* im = img ? img : v.bigimg;
            AO_CUDA(launch_sh_big(g, w, ph, api, stride, ks, v.scratch, make_plan(g).scratch, im, st), "sh_big");
            if (nz.on) AO_CUDA(launch_noise(g, w, im, step0 + c0, ks, nz, st), "noise");
            if (slp) AO_CUDA(launch_centroids(g, w, im, ks * (int)n_sel, slp, st), "centroids");
        }
    }
    return AO_OK;
}

static int run_psf(ao_geometry* g, const float* phase_dev, int64_t step0, int n_steps, double dt,
                   float* psf, int accumulate, cudaStream_t st, bool poly = false)
{
    if (g->sci.src.empty() || !g->psf_fft) return fail(AO_ERR_INVALID_ARG, "no science direction / psf_fft == 0");
    if (poly && g->band.n == 0) return fail(AO_ERR_INVALID_ARG, "ao_psf_poly: no wavelength band set (ao_set_psf_band)");
    if (!g->ws || g->ws_chunk < 1) return fail(AO_ERR_WORKSPACE, "ao_psf needs a workspace: call ao_set_workspace");
    const WsView v = ws_view(g);
    if (n_steps == 0 && !accumulate) {
        AO_CUDA(cudaMemsetAsync(psf, 0, sizeof(float) * g->sci.src.size() * (size_t)g->psf_fft * g->psf_fft, st), "memset");
        return AO_OK;
    }
    for (int c0 = 0; c0 < n_steps; c0 += v.chunk) {
        const int ks = (n_steps - c0 < v.chunk) ? n_steps - c0 : v.chunk;
        const float* ph; bool api; long long stride;
        if (phase_dev) {
            ph = phase_dev + (size_t)c0 * g->phase_elems_per_step; api = true; stride = g->phase_elems_per_step;
        } else {
            AO_CUDA(launch_trace(g, g->sci, false, g->sci.stage_elems, step0 + c0, ks, dt, v.stage, st), "trace");
            ph = v.stage; api = false; stride = g->sci.stage_elems;
        }
        const int kc = psf_chunk_steps(g);
        for (int k = 0; k < ks; k += kc) {
            const int kn = ks - k < kc ? ks - k : kc;
            if (poly) {
                for (int j = 0; j < g->band.n; ++j)
                    AO_CUDA(launch_psf_poly(g, ph + (size_t)k * stride, api, stride, kn, j, v.scratch, psf,
                                            (accumulate || c0 + k > 0 || j > 0) ? 1 : 0, st), "psf_poly");
            } else
            AO_CUDA(launch_psf(g, ph + (size_t)k * stride, api, stride, kn, v.scratch, psf,
                               (accumulate || c0 + k > 0) ? 1 : 0, st), "psf");
        }
    }
    return AO_OK;
}

}  // namespace ao

using namespace ao;

extern "C" {

const char* ao_last_error(void) { return g_err.c_str(); }
const char* ao_version(void)
{
#ifdef AO_PROFILE_SWITCHES
    return "ao-forward-b200 0.2 (sm_100a; PROFILING build: AO_DBG component switches compiled in, not for results)";
#else
    return "ao-forward-b200 0.2 (sm_100a; normal build)";
#endif
}

int ao_geometry_create(const ao_pupil* pupil, const ao_wfs* wfs, int n_wfs, const ao_layer* layers,
                       int n_layers, const ao_source* src, int n_src, double lambda_ref_m, int psf_fft,
                       ao_geometry** out)
{
    if (out) *out = nullptr;
    if (!out || !pupil || !pupil->amp_host || n_wfs < 0 || n_layers < 0 || n_src < 0 ||
        (n_wfs > 0 && !wfs) || (n_layers > 0 && !layers) || (n_src > 0 && !src))
        return fail(AO_ERR_INVALID_ARG, "ao_geometry_create: NULL pointer or negative count");
    if (pupil->n <= 0 || !(pupil->pitch_m > 0) || !(lambda_ref_m > 0))
        return fail(AO_ERR_SHAPE, "pupil n, pitch and lambda_ref must be positive");
    if (n_layers > kMaxLayers) return fail(AO_ERR_UNSUPPORTED, "more than 128 layers");
    for (int i = 0; i < n_wfs; ++i) {
        const ao_wfs& w = wfs[i];
        if (!w.amp_host) return fail(AO_ERR_INVALID_ARG, "wfs amp_host is NULL");
        if (w.n_sub <= 0 || w.n_samp <= 0 || w.fft <= 0 || w.bin <= 0 || w.n_pix <= 0 || w.n_samp > w.fft ||
            (w.fft & 1) || w.bin * w.n_pix > w.fft || ((w.fft - w.bin * w.n_pix) & 1))
            return fail(AO_ERR_SHAPE, "wfs: need n_samp <= fft, fft even, bin*n_pix <= fft, (fft-bin*n_pix) even");
        if (w.fft > 64) {
            if (!is_pow2(w.fft) || w.fft > 4096) return fail(AO_ERR_UNSUPPORTED, "wfs fft > 64 must be a power of two <= 4096");
            if ((size_t)w.bin * w.fft * sizeof(float2) > 200 * 1024)
                return fail(AO_ERR_UNSUPPORTED, "wfs fft > 64: bin*fft*8 bytes must fit in 200 KB of shared memory");
        }
        if ((size_t)w.n_sub * w.n_sub > 65535u * 32u) return fail(AO_ERR_UNSUPPORTED, "too many subapertures");
    }
    for (int i = 0; i < n_layers; ++i) {
        if (layers[i].n <= 1 || !(layers[i].pitch_m > 0)) return fail(AO_ERR_SHAPE, "layer n > 1 and pitch > 0 required");
        if (!layers[i].screen_dev) return fail(AO_ERR_INVALID_ARG, "layer screen_dev is NULL");
    }
    for (int i = 0; i < n_src; ++i) {
        if (src[i].wfs_index < -1 || src[i].wfs_index >= n_wfs) return fail(AO_ERR_INVALID_ARG, "source wfs_index out of range");
        if (!(src[i].lambda_m > 0) || !(src[i].altitude_m > 0)) return fail(AO_ERR_SHAPE, "source lambda and altitude must be positive");
    }
    if (psf_fft != 0 && (!is_pow2(psf_fft) || psf_fft < 64 || psf_fft > 4096 || psf_fft < pupil->n))
        return fail(AO_ERR_UNSUPPORTED, "psf_fft must be 0 or a power of two in [64, 4096] and >= pupil n");

    int dev_count = 0;
    AO_CUDA(cudaGetDeviceCount(&dev_count), "cudaGetDeviceCount");
    if (dev_count <= 0) return fail(AO_ERR_CUDA, "no CUDA device");

    ao_geometry* g = new ao_geometry();
    cudaError_t e = cudaSuccess;
    auto bail = [&](const char* what) { int rc = cuda_fail(e, what); destroy(g); return rc; };
    int dev = 0;
    cudaGetDevice(&dev);
    g->device = dev;
    cudaDeviceGetAttribute(&g->sm_count, cudaDevAttrMultiProcessorCount, dev);
    g->Np = pupil->n; g->pitch = pupil->pitch_m; g->lambda_ref = lambda_ref_m;
    const size_t np2 = (size_t)g->Np * g->Np;
    for (size_t i = 0; i < np2; ++i) { g->sumA2 += (double)pupil->amp_host[i] * pupil->amp_host[i]; g->sumA += (double)pupil->amp_host[i]; }
    if ((e = upload(&g->d_pupil_amp, pupil->amp_host, np2)) != cudaSuccess) return bail("pupil upload");

    const double PI = 3.14159265358979323846;
    g->layers.resize(n_layers);
    for (int i = 0; i < n_layers; ++i) {
        LayerP& lp = g->layers[i];
        lp.screen = layers[i].screen_dev; lp.S = layers[i].n;
        lp.mask = is_pow2(lp.S) ? lp.S - 1 : -1;
        lp.inv_pitch = 1.0 / layers[i].pitch_m; lp.height = layers[i].height_m;
        lp.wx = layers[i].wind_x_mps; lp.wy = layers[i].wind_y_mps;
    }
    if ((e = upload(&g->d_layers, g->layers.data(), g->layers.size())) != cudaSuccess) return bail("layers upload");

    g->wfs.resize(n_wfs);
    for (int i = 0; i < n_wfs; ++i) {
        WfsH& w = g->wfs[i];
        w.n_sub = wfs[i].n_sub; w.n = wfs[i].n_samp; w.M = wfs[i].fft; w.beta = wfs[i].bin; w.P = wfs[i].n_pix;
        w.min_illum = wfs[i].min_illum; w.logM = ilog2(w.M);
        // M > 64: two-pass HBM/L2 FFT.  M = 64 (c4's largest sweep point, n = 32: no fused kernel) is grouped with
        // them: one CTA per subaperture with both passes in shared memory (k_sh_mid64), same tables, no scratch.
        w.big = w.M >= 64;
        const int N = w.n_sub * w.n;
        const float* A = wfs[i].amp_host;
        w.valid.assign((size_t)w.n_sub * w.n_sub, 0);
        for (int p = 0; p < w.n_sub; ++p)
            for (int q = 0; q < w.n_sub; ++q) {
                double s = 0;
                for (int a = 0; a < w.n; ++a)
                    for (int b = 0; b < w.n; ++b) { const double v = A[(size_t)(p * w.n + a) * N + q * w.n + b]; s += v * v; }
                const bool ok = s / ((double)w.n * w.n) >= (double)w.min_illum;
                w.valid[(size_t)p * w.n_sub + q] = ok; w.n_valid += ok;
            }
        if ((e = upload(&w.d_amp, A, (size_t)N * N)) != cudaSuccess) return bail("wfs amp upload");
        if ((e = upload(&w.d_valid, w.valid.data(), w.valid.size())) != cudaSuccess) return bail("wfs valid upload");
        fused_tile_shape(w.M, &w.fused_G, &w.fused_R2);
        if (w.fused_G > 0) {
            // work items of the fused kernel: for each band of fused_R2 subaperture rows, runs of at most
            // fused_G adjacent columns in which at least one subaperture of the band is valid
            std::vector<int> items;
            for (int p = 0; p < w.n_sub; p += w.fused_R2) {
                auto need = [&](int q) {
                    for (int h = 0; h < w.fused_R2 && p + h < w.n_sub; ++h)
                        if (w.valid[(size_t)(p + h) * w.n_sub + q]) return true;
                    return false;
                };
                int q = 0;
                while (q < w.n_sub) {
                    if (!need(q)) { ++q; continue; }
                    int cnt = 0;
                    while (q + cnt < w.n_sub && cnt < w.fused_G && need(q + cnt)) ++cnt;
                    items.push_back(p); items.push_back(q); items.push_back(cnt); items.push_back(0);
                    q += cnt;
                }
            }
            w.n_fused_items = (int)(items.size() / 4);
            int* d = nullptr;
            if ((e = upload(&d, items.data(), items.size())) != cudaSuccess) return bail("fused items upload");
            w.fused_items = d;
            if (n_layers > 0 && (e = cudaMalloc((void**)&w.d_tmaps, (size_t)n_layers * (128 + sizeof(int2)))) != cudaSuccess) return bail("tensor map table");
        }
        if (w.M <= 64) {      // direct-DFT table of k_sh_generic (M = 64 uses it for extended beacons only)
            std::vector<float2> t(2 * w.M);
            for (int q = 0; q < 2 * w.M; ++q) t[q] = make_float2((float)cos(PI * q / w.M), (float)(-sin(PI * q / w.M)));
            if ((e = upload(&w.d_w2m, t.data(), t.size())) != cudaSuccess) return bail("twiddle upload");
        }
        if (w.big) {
            std::vector<float2> t(w.M / 2), pr(w.n);
            for (int k = 0; k < w.M / 2; ++k) t[k] = make_float2((float)cos(2 * PI * k / w.M), (float)(-sin(2 * PI * k / w.M)));
            for (int a = 0; a < w.n; ++a) {
                const long long q = ((long long)(w.M - 1) * a) % (2LL * w.M);     // exp(+i pi (M-1) a / M)
                pr[a] = make_float2((float)cos(PI * (double)q / w.M), (float)sin(PI * (double)q / w.M));
            }
            if ((e = upload(&w.d_tw, t.data(), t.size())) != cudaSuccess) return bail("twiddle upload");
            std::vector<float2> tf(w.M);
            for (int k = 0; k < w.M; ++k) tf[k] = make_float2((float)cos(2 * PI * k / w.M), (float)(-sin(2 * PI * k / w.M)));
            if ((e = upload(&w.d_twf, tf.data(), tf.size())) != cudaSuccess) return bail("twiddle upload");
            if ((e = upload(&w.d_pre, pr.data(), pr.size())) != cudaSuccess) return bail("pre-twiddle upload");
        }
    }

    g->sources.resize(n_src);
    long long off = 0;
    const double width = (double)g->Np * g->pitch;
    for (int i = 0; i < n_src; ++i) {
        SourceP& sp = g->sources[i];
        sp.wfs = src[i].wfs_index;
        sp.N = sp.wfs < 0 ? g->Np : g->wfs[sp.wfs].n_sub * g->wfs[sp.wfs].n;
        sp.d = width / (double)sp.N;
        sp.thx = src[i].theta_x_rad; sp.thy = src[i].theta_y_rad;
        sp.H = src[i].altitude_m; sp.inv_H = std::isinf(sp.H) ? 0.0 : 1.0 / sp.H;
        sp.scale = lambda_ref_m / src[i].lambda_m;
        sp.phase_off = off;
        sp.map = nullptr;
        off += (long long)sp.N * sp.N;
        g->all.src.push_back(i);
        if (sp.wfs < 0) g->sci.src.push_back(i); else g->wfs[sp.wfs].grp.src.push_back(i);
    }
    g->phase_elems_per_step = off;
    if ((e = upload(&g->d_sources, g->sources.data(), g->sources.size())) != cudaSuccess) return bail("sources upload");
    if ((e = build_group(g, g->all)) != cudaSuccess) return bail("group upload");
    if ((e = build_group(g, g->sci)) != cudaSuccess) return bail("group upload");
    for (auto& w : g->wfs) if ((e = build_group(g, w.grp)) != cudaSuccess) return bail("group upload");
    for (auto& w : g->wfs)      // two-pass FFT sensors put (source, subaperture) on gridDim.y
        if (w.M > 64 && w.grp.src.size() * (size_t)w.n_sub * w.n_sub > 65535u) {
            destroy(g);
            return fail(AO_ERR_UNSUPPORTED, "wfs fft > 64: sources x subapertures of one sensor must not exceed 65535");
        }

    g->psf_fft = psf_fft;
    if (psf_fft) {
        g->psf_log = ilog2(psf_fft);
        std::vector<float2> t(psf_fft), pr(g->Np);
        for (int k = 0; k < psf_fft; ++k) t[k] = make_float2((float)cos(2 * PI * k / psf_fft), (float)(-sin(2 * PI * k / psf_fft)));
        for (int a = 0; a < g->Np; ++a) pr[a] = make_float2((a & 1) ? -1.0f : 1.0f, 0.0f);
        if ((e = upload(&g->d_psf_tw, t.data(), t.size())) != cudaSuccess) return bail("psf twiddle upload");
        if ((e = upload(&g->d_psf_pre, pr.data(), pr.size())) != cudaSuccess) return bail("psf pre upload");
    }
    *out = g;
    return AO_OK;
}

int ao_geometry_destroy(ao_geometry* g)
{
    if (!g) return AO_OK;
    cudaDeviceSynchronize();
    destroy(g);
    return AO_OK;
}

size_t ao_workspace_bytes(const ao_geometry* g, int max_steps)
{
    if (!g) return 0;
    if (max_steps < 1) max_steps = 1;
    const Plan p = make_plan(g);
    const size_t per = p.per_step();
    size_t chunk = (size_t)max_steps;
    const size_t cap = (size_t)1 << 30;                      // keep the per-chunk staging near 1 GiB
    if (per > 0 && chunk * per > cap) chunk = cap / per > 0 ? cap / per : 1;
    return p.scratch + p.fixed + chunk * per + 256;
}

int ao_set_workspace(ao_geometry* g, void* workspace_dev, size_t bytes)
{
    if (!g) return fail(AO_ERR_INVALID_ARG, "NULL handle");
    g->ws = nullptr; g->ws_bytes = 0; g->ws_chunk = 0;
    if (!workspace_dev) return AO_OK;
    if (((uintptr_t)workspace_dev & 255) != 0) return fail(AO_ERR_INVALID_ARG, "workspace must be 256-byte aligned");
    const Plan p = make_plan(g);
    const size_t base = p.scratch + p.fixed, per = p.per_step();
    if (bytes < base + per) return fail(AO_ERR_WORKSPACE, "workspace smaller than ao_workspace_bytes(g, 1)");
    g->ws = (char*)workspace_dev; g->ws_bytes = bytes;
    const size_t c = per ? (bytes - base) / per : 1u << 20;
    g->ws_chunk = (int)(c > (1u << 20) ? (1u << 20) : c);
    return AO_OK;
}

size_t ao_phase_elems_per_step(const ao_geometry* g) { return g ? (size_t)g->phase_elems_per_step : 0; }

size_t ao_phase_offset(const ao_geometry* g, int source, int step)
{
    if (!g || source < 0 || source >= (int)g->sources.size() || step < 0) return (size_t)-1;
    return (size_t)step * (size_t)g->phase_elems_per_step + (size_t)g->sources[source].phase_off;
}

int ao_wfs_valid(const ao_geometry* g, int wfs_index, uint8_t* valid_host)
{
    if (!g || wfs_index < 0 || wfs_index >= (int)g->wfs.size()) return -1;
    const WfsH& w = g->wfs[wfs_index];
    if (valid_host) memcpy(valid_host, w.valid.data(), w.valid.size());
    return w.n_valid;
}

int64_t ao_launch_count(const ao_geometry* g) { return g ? g->launches : 0; }
uint64_t ao_last_h2d_bytes(const ao_geometry* g) { return g ? g->h2d_bytes : 0; }

int ao_trace_layers(ao_geometry* g, int64_t step0, int n_steps, double dt_s, float* phase_dev, void* cuda_stream)
{
    int rc = check_entry(g); if (rc) return rc;
    if (n_steps < 0) return fail(AO_ERR_INVALID_ARG, "ao_trace_layers: n_steps < 0");
    if (n_steps == 0) return AO_OK;
    if (!phase_dev) return fail(AO_ERR_INVALID_ARG, "ao_trace_layers: phase_dev is NULL");
    AO_CUDA(launch_trace(g, g->all, true, g->phase_elems_per_step, step0, n_steps, dt_s, phase_dev,
                         (cudaStream_t)cuda_stream), "trace");
    return AO_OK;
}

int ao_sh_images(ao_geometry* g, int wfs_index, const float* phase_dev, int64_t step0, int n_steps,
                 double dt_s, const ao_noise* noise, float* images_dev, float* slopes_dev, void* cuda_stream)
{
    int rc = check_entry(g); if (rc) return rc;
    if (wfs_index < 0 || wfs_index >= (int)g->wfs.size()) return fail(AO_ERR_INVALID_ARG, "ao_sh_images: wfs_index out of range");
    if (n_steps < 0) return fail(AO_ERR_INVALID_ARG, "ao_sh_images: n_steps < 0");
    if (n_steps == 0) return AO_OK;
    if (!images_dev && !slopes_dev) return fail(AO_ERR_INVALID_ARG, "ao_sh_images: no output buffer");
    return run_wfs(g, wfs_index, phase_dev, step0, n_steps, dt_s, noise, images_dev, slopes_dev, (cudaStream_t)cuda_stream);
}

int ao_centroids(ao_geometry* g, int wfs_index, const float* images_dev, int n_image_sets, float* slopes_dev,
                 void* cuda_stream)
{
    int rc = check_entry(g); if (rc) return rc;
    if (wfs_index < 0 || wfs_index >= (int)g->wfs.size()) return fail(AO_ERR_INVALID_ARG, "ao_centroids: wfs_index out of range");
    if (!images_dev || !slopes_dev || n_image_sets < 0) return fail(AO_ERR_INVALID_ARG, "ao_centroids: NULL buffer or negative count");
    AO_CUDA(launch_centroids(g, g->wfs[wfs_index], images_dev, n_image_sets, slopes_dev, (cudaStream_t)cuda_stream), "centroids");
    return AO_OK;
}

int ao_psf(ao_geometry* g, const float* phase_dev, int64_t step0, int n_steps, double dt_s, float* psf_dev,
           int accumulate, void* cuda_stream)
{
    int rc = check_entry(g); if (rc) return rc;
    if (!psf_dev || n_steps < 0) return fail(AO_ERR_INVALID_ARG, "ao_psf: psf_dev NULL or n_steps < 0");
    return run_psf(g, phase_dev, step0, n_steps, dt_s, psf_dev, accumulate, (cudaStream_t)cuda_stream);
}

// ao_forward_host: host -> device copy of the part of screen l that steps [step0, step0 + n_steps) read: the bounding box
// of the footprints of every source that sees the layer, at the first and the last step (the footprint moves linearly
// in time), plus a margin for the staged boxes of the tiled kernels (they load a few aligned columns and rows beyond the
// taps); periodic wrap splits the box in up to 2 x 2 pieces.  A box as large as the screen uploads the whole screen.
static int upload_screen_region(ao_geometry* g, int l, const float* host, int64_t step0, int n_steps, double dt, cudaStream_t st)
{
    const LayerP& lp = g->layers[l];
    const long long S = lp.S;
    const size_t pitch = sizeof(float) * (size_t)S;
    auto whole = [&]() {
        g->h2d_bytes += pitch * (size_t)S;
        return cudaMemcpyAsync((void*)lp.screen, host, pitch * (size_t)S, cudaMemcpyHostToDevice, st);
    };
    if (n_steps <= 0) return AO_OK;
    bool any = false;
    double umin = 0, umax = 0, vmin = 0, vmax = 0;
    for (const SourceP& sp : g->sources) {
        if (!(lp.height < sp.H)) continue;
        const double gamma = 1.0 - lp.height * sp.inv_H, x0 = -0.5 * (double)(sp.N - 1) * sp.d, c = 0.5 * (double)(S - 1);
        const double du = gamma * sp.d * lp.inv_pitch;
        for (int e = 0; e < 2; ++e) {
            const double t = (double)(step0 + (e ? n_steps - 1 : 0)) * dt;
            const double u0 = (gamma * x0 + lp.height * sp.thx - lp.wx * t) * lp.inv_pitch + c, u1 = u0 + (sp.N - 1) * du;
            const double v0 = (gamma * x0 + lp.height * sp.thy - lp.wy * t) * lp.inv_pitch + c, v1 = v0 + (sp.N - 1) * du;
            if (!any) { umin = std::min(u0, u1); umax = std::max(u0, u1); vmin = std::min(v0, v1); vmax = std::max(v0, v1); any = true; }
            umin = std::min(umin, std::min(u0, u1)); umax = std::max(umax, std::max(u0, u1));
            vmin = std::min(vmin, std::min(v0, v1)); vmax = std::max(vmax, std::max(v0, v1));
        }
    }
    if (!any) return AO_OK;                                   // no source sees this layer: nothing is read
    const long long margin = 24;
    const long long c_lo = (long long)floor(umin) - margin, c_hi = (long long)floor(umax) + 1 + margin;
    const long long r_lo = (long long)floor(vmin) - margin, r_hi = (long long)floor(vmax) + 1 + margin;
    const long long W = c_hi - c_lo + 1, H = r_hi - r_lo + 1;
    if (W >= S || H >= S || fabs(umin) > 1e15 || fabs(vmin) > 1e15) { AO_CUDA(whole(), "screen upload"); return AO_OK; }
    const long long cw = ((c_lo % S) + S) % S, rw = ((r_lo % S) + S) % S;
    const long long cpart[2][2] = {{cw, std::min(W, S - cw)}, {0, W - std::min(W, S - cw)}};      // {start, count}
    const long long rpart[2][2] = {{rw, std::min(H, S - rw)}, {0, H - std::min(H, S - rw)}};
    float* dev = const_cast<float*>(lp.screen);
    for (int a = 0; a < 2; ++a)
        for (int b = 0; b < 2; ++b) {
            const long long r0 = rpart[a][0], nr = rpart[a][1], c0 = cpart[b][0], nc = cpart[b][1];
            if (nr <= 0 || nc <= 0) continue;
            const size_t off = (size_t)r0 * S + (size_t)c0;
            AO_CUDA(cudaMemcpy2DAsync(dev + off, pitch, host + off, pitch, sizeof(float) * (size_t)nc, (size_t)nr,
                                      cudaMemcpyHostToDevice, st), "screen region upload");
            g->h2d_bytes += sizeof(float) * (size_t)nc * (size_t)nr;
        }
    return AO_OK;
}

// Shared by ao_forward and ao_forward_host: all WFS (slopes only) and the PSF for steps [step0, step0 + n_steps), in order
// on the caller's stream: the workspace users first (big-FFT sensors, PSF: many short launches), then the fused sensors.
// A library-owned high-priority side stream for the workspace users was measured and removed: the fused kernel's CTAs hold the
// whole register file of an SM, nothing overlaps, and the fork / join cost 4 us per step on c4 and 50 us per step on c3.
static int forward_chunk(ao_geometry* g, int64_t step0, int n_steps, double dt_s, const ao_noise* noise,
                         float* const* slopes, float* psf, int accumulate, cudaStream_t st)
{
    int rc = AO_OK;
    const bool want_psf = psf && g->psf_fft && !g->sci.src.empty();
    for (int pass = 0; pass < 2 && rc == AO_OK; ++pass) {
        for (size_t wi = 0; wi < g->wfs.size() && rc == AO_OK; ++wi) {
            const WfsH& w = g->wfs[wi];
            if (!slopes || !slopes[wi] || w.grp.src.empty()) continue;
            const bool fused = (!w.big || w.M == 64) && fused_supported(g, w, dt_s);
            if (fused != (pass == 1)) continue;
            rc = run_wfs(g, (int)wi, nullptr, step0, n_steps, dt_s, noise, nullptr, slopes[wi], st);
        }
        if (pass == 0 && want_psf && rc == AO_OK)
            rc = run_psf(g, nullptr, step0, n_steps, dt_s, psf, accumulate, st, g->band.n > 0);
    }
    return rc;
}

int ao_set_phase_map(ao_geometry* g, int source, const float* map_dev)
{
    int rc = check_entry(g); if (rc) return rc;
    if (source < 0 || source >= (int)g->sources.size()) return fail(AO_ERR_INVALID_ARG, "ao_set_phase_map: bad source index");
    AO_CUDA(cudaDeviceSynchronize(), "synchronize before the source table update");
    g->sources[source].map = map_dev;
    AO_CUDA(cudaMemcpy(g->d_sources + source, &g->sources[source], sizeof(SourceP), cudaMemcpyHostToDevice), "source table update");
    return AO_OK;
}

// radix-2 FFT in FP64 on the host (tables of the chirp-z transform only)
static void host_fft(std::vector<std::complex<double>>& x)
{
    const size_t n = x.size();
    for (size_t i = 1, j = 0; i < n; ++i) {
        size_t bit = n >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) std::swap(x[i], x[j]);
    }
    const double PI = 3.14159265358979323846;
    for (size_t len = 2; len <= n; len <<= 1)
        for (size_t base = 0; base < n; base += len)
            for (size_t k = 0; k < len / 2; ++k) {
                const std::complex<double> w = std::polar(1.0, -2.0 * PI * (double)k / (double)len);
                const std::complex<double> u = x[base + k], t = w * x[base + k + len / 2];
                x[base + k] = u + t; x[base + k + len / 2] = u - t;
            }
}

int ao_set_psf_band(ao_geometry* g, const double* lambdas_m_host, const double* weights_host, int n_lambda)
{
    int rc = check_entry(g); if (rc) return rc;
    if (n_lambda < 0 || n_lambda > 256 || (n_lambda > 0 && (!lambdas_m_host || !weights_host)))
        return fail(AO_ERR_INVALID_ARG, "ao_set_psf_band: need 0 <= n_lambda <= 256 and non-NULL arrays");
    if (n_lambda > 0 && (g->sci.src.empty() || !g->psf_fft)) return fail(AO_ERR_INVALID_ARG, "ao_set_psf_band: no science direction / psf_fft == 0");
    const int M = g->psf_fft, Np = g->Np;
    int logL = 8;
    while ((1 << logL) < M + Np - 1) ++logL;
    if (n_lambda > 0 && logL > 12) return fail(AO_ERR_UNSUPPORTED, "ao_set_psf_band: psf_fft + pupil n - 1 must not exceed 4096");
    double lambda_s = 0.0;
    for (size_t i = 0; i < g->sci.src.size() && n_lambda > 0; ++i) {
        const double l = g->lambda_ref / g->sources[g->sci.src[i]].scale;
        if (i == 0) lambda_s = l;
        else if (fabs(l - lambda_s) > 1e-12 * lambda_s) return fail(AO_ERR_UNSUPPORTED, "ao_set_psf_band: the science directions must share one wavelength");
    }
    for (int j = 0; j < n_lambda; ++j)
        if (!(lambdas_m_host[j] > 0)) return fail(AO_ERR_INVALID_ARG, "ao_set_psf_band: wavelengths must be positive");
    AO_CUDA(cudaDeviceSynchronize(), "synchronize before the band table update");
    free_band(g);
    if (n_lambda == 0) return AO_OK;
    const int L = 1 << logL;
    const double PI = 3.14159265358979323846;
    auto cis_turns = [&](double t) { t -= floor(t); return std::polar(1.0, 2.0 * PI * t); };     // exp(2 pi i t), reduced in FP64
    std::vector<float2> tw(L), cin((size_t)n_lambda * Np), Hf((size_t)n_lambda * L), cout((size_t)n_lambda * M);
    for (int k = 0; k < L; ++k) tw[k] = make_float2((float)cos(2 * PI * k / L), (float)(-sin(2 * PI * k / L)));
    PsfBand B;
    B.n = n_lambda; B.L = L; B.logL = logL;
    for (int j = 0; j < n_lambda; ++j) {
        const double s = lambda_s / lambdas_m_host[j];
        B.scale.push_back(s); B.weight.push_back(weights_host[j]);
        for (int b = 0; b < Np; ++b) {          // exp(-i pi s b^2 / M) = exp(2 pi i (-s b^2 / (2M)))
            const std::complex<double> c = cis_turns(-s * (double)b * b / (2.0 * M));
            cin[(size_t)j * Np + b] = make_float2((float)c.real(), (float)c.imag());
        }
        for (int k = 0; k < M; ++k) {
            const double kap = (double)k - 0.5 * M;
            const std::complex<double> c = cis_turns(-s * kap * kap / (2.0 * M));
            cout[(size_t)j * M + k] = make_float2((float)c.real(), (float)c.imag());
        }
        std::vector<std::complex<double>> h(L, 0.0);
        for (int u = -(Np - 1); u <= M - 1; ++u) {
            const double t = (double)u - 0.5 * M;
            h[(size_t)((u % L + L) % L)] = cis_turns(s * t * t / (2.0 * M));
        }
        host_fft(h);
        for (int i = 0; i < L; ++i) Hf[(size_t)j * L + i] = make_float2((float)(h[i].real() / L), (float)(h[i].imag() / L));
    }
    cudaError_t e = upload(&B.d_tw, tw.data(), tw.size());
    if (e == cudaSuccess) e = upload(&B.d_cin, cin.data(), cin.size());
    if (e == cudaSuccess) e = upload(&B.d_Hf, Hf.data(), Hf.size());
    if (e == cudaSuccess) e = upload(&B.d_cout, cout.data(), cout.size());
    g->band = B;
    if (e != cudaSuccess) { free_band(g); return cuda_fail(e, "band table upload"); }
    return AO_OK;
}

int ao_psf_poly(ao_geometry* g, const float* phase_dev, int64_t step0, int n_steps, double dt_s, float* psf_dev,
                int accumulate, void* cuda_stream)
{
    int rc = check_entry(g); if (rc) return rc;
    if (!psf_dev || n_steps < 0) return fail(AO_ERR_INVALID_ARG, "ao_psf_poly: psf_dev NULL or n_steps < 0");
    return run_psf(g, phase_dev, step0, n_steps, dt_s, psf_dev, accumulate, (cudaStream_t)cuda_stream, true);
}

int ao_set_sodium(ao_geometry* g, int wfs_index, int n_z, const double* z_m_host, const double* rho_host, int n_t,
                  const double* launch_xy_m_host)
{
    int rc = check_entry(g); if (rc) return rc;
    if (wfs_index < 0 || wfs_index >= (int)g->wfs.size()) return fail(AO_ERR_INVALID_ARG, "ao_set_sodium: wfs_index out of range");
    WfsH& w = g->wfs[wfs_index];
    if (n_z < 0 || n_z > 64 || (n_z > 0 && (n_t < 1 || !z_m_host || !rho_host || !launch_xy_m_host)))
        return fail(AO_ERR_INVALID_ARG, "ao_set_sodium: need 0 <= n_z <= 64 and, for n_z > 0, n_t >= 1 and non-NULL arrays");
    if (n_z > 0 && w.M > 64) return fail(AO_ERR_UNSUPPORTED, "ao_set_sodium: extended beacons are implemented for sensors with fft <= 64");
    const size_t n_sel = w.grp.src.size();
    std::vector<double> gt(n_sel * (size_t)n_z);
    for (size_t si = 0; si < n_sel && n_z > 0; ++si) {
        const SourceP& sp = g->sources[w.grp.src[si]];
        const double lambda_s = g->lambda_ref / sp.scale;
        if (std::isinf(sp.H)) return fail(AO_ERR_INVALID_ARG, "ao_set_sodium: a source of this sensor is at infinity");
        for (int iz = 0; iz < n_z; ++iz) {
            if (!(z_m_host[iz] > 0)) return fail(AO_ERR_INVALID_ARG, "ao_set_sodium: altitudes must be positive");
            gt[si * n_z + iz] = (1.0 / sp.H - 1.0 / z_m_host[iz]) * sp.d / lambda_s;
        }
    }
    AO_CUDA(cudaDeviceSynchronize(), "synchronize before the sodium table update");
    free_sodium(w);
    if (n_z == 0) return AO_OK;
    std::vector<float> rho((size_t)n_t * n_z);
    for (size_t i = 0; i < rho.size(); ++i) rho[i] = (float)rho_host[i];
    float* d_rho = nullptr; double* d_g = nullptr; double* d_l = nullptr;
    cudaError_t e = upload(&d_rho, rho.data(), rho.size());
    if (e == cudaSuccess) e = upload(&d_g, gt.data(), gt.size());
    if (e == cudaSuccess) e = upload(&d_l, launch_xy_m_host, 2 * n_sel);
    if (e != cudaSuccess) { cudaFree(d_rho); cudaFree(d_g); cudaFree(d_l); return cuda_fail(e, "sodium table upload"); }
    w.na.n_z = n_z; w.na.n_t = n_t; w.na.rho = d_rho; w.na.gturn = d_g; w.na.launch = d_l;
    return AO_OK;
}

int ao_modes_to_map(ao_geometry* g, const float* modes_dev, int n_modes, long long n_elems,
                    const float* coeffs_dev, float sign, float* map_dev, void* cuda_stream)
{
    int rc = check_entry(g); if (rc) return rc;
    if (n_modes < 0 || n_elems < 0) return fail(AO_ERR_INVALID_ARG, "ao_modes_to_map: negative size");
    if (!map_dev || (n_modes > 0 && (!modes_dev || !coeffs_dev))) return fail(AO_ERR_INVALID_ARG, "ao_modes_to_map: NULL pointer");
    AO_CUDA(launch_modes_to_map(g, modes_dev, n_modes, n_elems, coeffs_dev, sign, map_dev, (cudaStream_t)cuda_stream), "modes_to_map");
    return AO_OK;
}

int ao_strehl(ao_geometry* g, const float* psf_dev, double n_exposures, float* strehl_dev, void* cuda_stream)
{
    int rc = check_entry(g); if (rc) return rc;
    if (g->sci.src.empty() || !g->psf_fft) return fail(AO_ERR_INVALID_ARG, "ao_strehl: no science direction / psf_fft == 0");
    if (!psf_dev || !strehl_dev || !(n_exposures > 0.0)) return fail(AO_ERR_INVALID_ARG, "ao_strehl: NULL pointer or n_exposures <= 0");
    const double M = (double)g->psf_fft;
    const double peak_flat = g->sumA2 > 0 ? g->sumA * g->sumA / (M * M * g->sumA2) : 0.0;
    const float inv = peak_flat > 0 ? (float)(1.0 / (n_exposures * peak_flat)) : 0.0f;
    AO_CUDA(launch_strehl(g, psf_dev, (int)g->sci.src.size(), g->psf_fft, inv, strehl_dev, (cudaStream_t)cuda_stream), "strehl");
    return AO_OK;
}

int ao_strehl_marechal(ao_geometry* g, const float* phase_dev, int n_steps, float* strehl_dev, void* cuda_stream)
{
    int rc = check_entry(g); if (rc) return rc;
    if (g->sci.src.empty()) return fail(AO_ERR_INVALID_ARG, "ao_strehl_marechal: no science direction");
    if (!phase_dev || !strehl_dev || n_steps < 0) return fail(AO_ERR_INVALID_ARG, "ao_strehl_marechal: NULL pointer or n_steps < 0");
    AO_CUDA(launch_marechal(g, phase_dev, g->phase_elems_per_step, n_steps, strehl_dev, (cudaStream_t)cuda_stream), "marechal");
    return AO_OK;
}

int ao_forward(ao_geometry* g, int64_t step0, int n_steps, double dt_s, const ao_noise* noise,
               float* const* slopes_dev, float* psf_dev, int accumulate, void* cuda_stream)
{
    int rc = check_entry(g); if (rc) return rc;
    if (n_steps < 0) return fail(AO_ERR_INVALID_ARG, "ao_forward: n_steps < 0");
    return forward_chunk(g, step0, n_steps, dt_s, noise, slopes_dev, psf_dev, accumulate, (cudaStream_t)cuda_stream);
}

int ao_forward_host(ao_geometry* g, const float* const* screens_host, int64_t step0, int n_steps, double dt_s,
                    const ao_noise* noise, float* const* slopes_host, float* psf_host, void* cuda_stream)
{
    int rc = check_entry(g); if (rc) return rc;
    if (n_steps < 0) return fail(AO_ERR_INVALID_ARG, "ao_forward_host: n_steps < 0");
    if (!g->ws || g->ws_chunk < 1) return fail(AO_ERR_WORKSPACE, "ao_forward_host needs a workspace");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    g->h2d_bytes = 0;
    if (screens_host)
        for (size_t l = 0; l < g->layers.size(); ++l) {
            if (!screens_host[l]) return fail(AO_ERR_INVALID_ARG, "ao_forward_host: screens_host[l] is NULL");
            rc = upload_screen_region(g, (int)l, screens_host[l], step0, n_steps, dt_s, st);
            if (rc) return rc;
        }
    const WsView v = ws_view(g);
    const bool want_psf = psf_host && g->psf_fft && !g->sci.src.empty();
    if (n_steps == 0 && want_psf) { rc = run_psf(g, nullptr, step0, 0, dt_s, v.psf_stage, 0, st); if (rc) return rc; }
    std::vector<float*> dst(g->wfs.size(), nullptr);
    for (int c0 = 0; c0 < n_steps; c0 += v.chunk) {
        const int ks = (n_steps - c0 < v.chunk) ? n_steps - c0 : v.chunk;
        char* sl = (char*)v.slopes;
        for (size_t wi = 0; wi < g->wfs.size(); ++wi) {
            const WfsH& w = g->wfs[wi];
            const size_t per = sizeof(float) * w.grp.src.size() * 2 * (size_t)w.n_sub * w.n_sub;
            dst[wi] = (slopes_host && slopes_host[wi] && !w.grp.src.empty()) ? (float*)sl : nullptr;
            sl += align256(per) * (size_t)v.chunk;
        }
        rc = forward_chunk(g, step0 + c0, ks, dt_s, noise, dst.data(), want_psf ? v.psf_stage : nullptr, c0 > 0 ? 1 : 0, st);
        if (rc) return rc;
        for (size_t wi = 0; wi < g->wfs.size(); ++wi) {
            if (!dst[wi]) continue;
            const WfsH& w = g->wfs[wi];
            const size_t per = sizeof(float) * w.grp.src.size() * 2 * (size_t)w.n_sub * w.n_sub;
            AO_CUDA(cudaMemcpyAsync((char*)slopes_host[wi] + per * (size_t)c0, dst[wi], per * (size_t)ks,
                                    cudaMemcpyDeviceToHost, st), "slopes download");
        }
    }
    if (want_psf)
        AO_CUDA(cudaMemcpyAsync(psf_host, v.psf_stage, sizeof(float) * g->sci.src.size() * (size_t)g->psf_fft * g->psf_fft,
                                cudaMemcpyDeviceToHost, st), "psf download");
    AO_CUDA(cudaStreamSynchronize(st), "stream synchronize");
    return AO_OK;
}

}  // extern "C"
