// ao_internal.cuh -- internal declarations of libao.so (CUDA path only; the oracle shares nothing with it).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string>
#include <vector>

#include "ao.h"

namespace ao {

constexpr int kMaxLayers = 128;

// Per-layer parameters in device memory (one array per handle).
struct LayerP {
    const float* screen;   // [S][S]
    int S;
    int mask;              // S-1 if S is a power of two, else -1 (use %)
    double inv_pitch;      // 1/d_l
    double height;         // h_l
    double wx, wy;         // wind m/s
};

// Per-source parameters in device memory.
struct SourceP {
    int N;                 // grid samples per side
    int wfs;               // wfs index or -1
    double d;              // grid pitch d_s
    double thx, thy;       // direction (rad)
    double H;              // altitude (inf for NGS/science)
    double inv_H;          // 1/H (0 for inf)
    double scale;          // lambda_ref / lambda_s
    long long phase_off;   // element offset inside one step of the caller's phase buffer
    const float* map;      // additive phase map [N][N], radians at the source's wavelength, or NULL (ao_set_phase_map)
};

// A group of sources processed together (all / those of one WFS / science directions).
struct Group {
    std::vector<int> src;          // global source indices, ascending
    int* d_src = nullptr;          // device copy
    long long* d_off_api = nullptr;   // phase offsets in the API layout (per member)
    long long* d_off_stage = nullptr; // phase offsets in the compact staging layout (per member)
    long long stage_elems = 0;     // elements per step in the staging layout
    int max_N = 0;
};

struct NoiseP {
    int on;
    uint32_t key0, key1;
    float photons, read_noise;
};

// Extended sodium layer of the LGS sensors of one WFS (ao_set_sodium; DESIGN.md section 3 reading O9).
struct SodiumP {
    int n_z = 0, n_t = 0;              // scatterers per profile, time samples of the profile (0: point beacon)
    const float* rho = nullptr;        // [n_t][n_z] weights, device
    const double* gturn = nullptr;     // [n_sel][n_z]: (1/H_s - 1/z) d_s / lambda_s, turns per sample per metre of baseline
    const double* launch = nullptr;    // [n_sel][2] launch point, metres in the pupil plane
};

// Spot shift of one scatterer as a phase ramp in 0.32 fixed-point turns per sample (exact wrap-around arithmetic).
struct ElongRamp { uint32_t fx, fy; };

struct WfsH {
    int n_sub, n, M, beta, P;
    float min_illum;
    bool big;                       // M > 64: multi-pass HBM FFT
    int logM = 0;
    float* d_amp = nullptr;         // [N][N]
    uint8_t* d_valid = nullptr;     // [n_sub^2]
    std::vector<uint8_t> valid;
    int n_valid = 0;
    float2* d_w2m = nullptr;        // W[q] = exp(-i pi q / M), q < 2M     (small path)
    float2* d_tw = nullptr;         // exp(-2 pi i k / M), k < M/2         (big path, generic fallback)
    float2* d_twf = nullptr;        // exp(-2 pi i k / M), k < M           (big path, Stockham passes)
    float2* d_pre = nullptr;        // pre-twiddle exp(+i pi (M-1) a / M), a < n  (big path)
    SodiumP na;                     // extended beacon (device pointers owned by the handle), n_z = 0: none
    unsigned char* d_tmaps = nullptr;   // CUtensorMap[n_layers] of the fused kernel's staged boxes (device), see k_fused.cu
    int tm_pitch = 0, tm_rows = 0;      // plan the maps were encoded for (0: not encoded yet)
    double tm_dt = 0.0;
    void* fused_items = nullptr;    // device WorkItem[]: runs of <= fused_G adjacent valid subapertures
    int n_fused_items = 0, fused_G = 0, fused_R2 = 0;
    Group grp;
};

// Wavelength band of the polychromatic science PSF (ao_set_psf_band; reading O8): chirp-z tables per wavelength.
struct PsfBand {
    int n = 0, L = 0, logL = 0;             // wavelengths, FFT length of the circular convolution (>= M + Np - 1)
    std::vector<double> scale, weight;      // s_j = lambda_s / lambda_j, w_j
    float2* d_tw = nullptr;                 // exp(-2 pi i k / L), k < L
    float2* d_cin = nullptr;                // [n][Np]  exp(-i pi s b^2 / M)
    float2* d_Hf = nullptr;                 // [n][L]   FFT_L(h) / L, h[u] = exp(+i pi s (u - M/2)^2 / M)
    float2* d_cout = nullptr;               // [n][M]   exp(-i pi s (k' - M/2)^2 / M)
};

}  // namespace ao

struct ao_geometry {
    int Np = 0;
    double pitch = 0;
    float* d_pupil_amp = nullptr;
    double sumA2 = 0, sumA = 0;
    std::vector<ao::WfsH> wfs;
    std::vector<ao::LayerP> layers;
    ao::LayerP* d_layers = nullptr;
    std::vector<ao::SourceP> sources;
    ao::SourceP* d_sources = nullptr;
    double lambda_ref = 0;
    int psf_fft = 0, psf_log = 0;
    float2* d_psf_tw = nullptr;       // exp(-2 pi i k / M), k < M
    float2* d_psf_pre = nullptr;      // (-1)^a as a complex table, a < Np
    ao::Group all, sci;
    ao::PsfBand band;                 // n = 0: no band set
    long long phase_elems_per_step = 0;
    // workspace
    char* ws = nullptr;
    size_t ws_bytes = 0;
    int ws_chunk = 0;                 // steps per internal chunk that fit the workspace
    int64_t launches = 0;
    uint64_t h2d_bytes = 0;           // bytes of screens uploaded by the last ao_forward_host
    int sm_count = 148;
    int device = 0;                   // the CUDA device the handle was created on (made current by every call)
};

namespace ao {

// ---- kernel launchers (each returns the cudaError of the launch) ----
cudaError_t launch_trace(ao_geometry* g, const Group& grp, bool api_layout, long long step_stride,
                         int64_t step0, int n_steps, double dt, float* phase, cudaStream_t st);

cudaError_t launch_sh_small(ao_geometry* g, const WfsH& w, const float* phase, bool api_layout,
                            long long step_stride, int64_t step0, int n_steps, const NoiseP& noise,
                            float* images, float* slopes, cudaStream_t st);

// in-register FFT path for M in {16, 24, 32}, n = M/2, full window (k_sh_reg.cu); other shapes: launch_sh_small
bool sh_reg_supported(const WfsH& w);
cudaError_t launch_sh_reg(ao_geometry* g, const WfsH& w, const float* phase, bool api_layout, long long step_stride,
                          int64_t step0, int n_steps, const NoiseP& noise, float* images, float* slopes, cudaStream_t st);

cudaError_t launch_centroids(ao_geometry* g, const WfsH& w, const float* images, int n_sets,
                             float* slopes, cudaStream_t st);

cudaError_t launch_modes_to_map(ao_geometry* g, const float* modes, int n_modes, long long n_elems, const float* coeffs,
                                float sign, float* map, cudaStream_t st);

cudaError_t launch_strehl(ao_geometry* g, const float* psf, int n_dir, int M, float inv_norm, float* strehl, cudaStream_t st);

cudaError_t launch_marechal(ao_geometry* g, const float* phase, long long step_stride, int n_steps, float* strehl,
                            cudaStream_t st);

cudaError_t launch_noise(ao_geometry* g, const WfsH& w, float* images, int64_t step0, int n_steps,
                         const NoiseP& noise, cudaStream_t st);

// big FFT: SH mode for one step-chunk of WFS w (images out); PSF mode for ks <= psf_chunk_steps(g)
// consecutive steps summed into psf (phase of step j at phase + j * step_stride).
cudaError_t launch_sh_big(ao_geometry* g, const WfsH& w, const float* phase, bool api_layout,
                          long long step_stride, int n_steps, float2* scratch, size_t scratch_bytes, float* images,
                          cudaStream_t st);
cudaError_t launch_psf(ao_geometry* g, const float* phase, bool api_layout, long long step_stride,
                       int ks, float2* scratch, float* psf, int accumulate, cudaStream_t st);
int psf_chunk_steps(const ao_geometry* g);
// polychromatic PSF: wavelength j of the band, ks <= psf_chunk_steps(g) steps added into psf (k_psf_poly.cu)
cudaError_t launch_psf_poly(ao_geometry* g, const float* phase, bool api_layout, long long step_stride, int ks,
                            int j, float2* scratch, float* psf, int accumulate, cudaStream_t st);
bool sh_big_fast(const WfsH& w);                                    // the Stockham two-pass path applies (else generic)

// fused trace + SH + CoG (k_fused.cu); cudaErrorNotSupported if the geometry is outside its fast path
bool fused_supported(const ao_geometry* g, const WfsH& w, double dt);
cudaError_t launch_fused(ao_geometry* g, const WfsH& w, int64_t step0, int n_steps, double dt,
                         const NoiseP& noise, float* images, float* slopes, cudaStream_t st);
void fused_tile_shape(int M, int* G, int* R2);
// tiled ray-trace into a phase buffer (k_fused.cu); cudaErrorNotSupported if outside its fast path
cudaError_t launch_trace_tiled(ao_geometry* g, const Group& grp, bool api_layout, long long step_stride,
                               int64_t step0, int n_steps, double dt, float* phase, cudaStream_t st);

size_t sh_big_scratch_bytes(const ao_geometry* g, const WfsH& w);   // per step
size_t psf_scratch_bytes(const ao_geometry* g);                      // per step (x psf_chunk_steps)

void set_error(const std::string& msg);

}  // namespace ao
