/* ao.h -- C ABI of libao.so: the per-time-step optical forward model of the MAORY
 * multi-conjugate adaptive-optics Monte-Carlo simulator (arxiv 1608.00386), B200 (sm_100a).
 *
 * Citations are "PAPER.md:<line> (section)" of /root/reference/PAPER.md.  The paper names
 * the operations but prints no formula; the numerical definitions are the readings listed
 * in DESIGN.md section 3 (taken from SURVEY.md section 8(c), O1..O7).
 *
 * Conventions
 *   - All arrays are row-major [y][x], x fastest, fp32 unless stated.
 *   - "_dev" pointers are CUDA device pointers, "_host" pointers are host pointers.
 *   - Grid (O1): sample j of an N-sample grid sits at x_j = (j-(N-1)/2) d.  The pupil grid has
 *     N_p samples of pitch d_p; the grid of WFS w has N_w = n_sub*n_samp samples spanning the
 *     same width (d_w = N_p d_p / N_w); a science direction uses the pupil grid.
 *   - Every call returns an ao_status; nothing throws or aborts across the ABI.  All argument
 *     and shape validation happens before any kernel is launched.  Compute calls are
 *     asynchronous on `cuda_stream` (a cudaStream_t passed as void*; NULL = default stream);
 *     a CUDA error raised by earlier asynchronous work is reported as AO_ERR_CUDA by the next
 *     call.  ao_last_error() returns a thread-local, never-NULL message for the last failure.
 *   - Ownership: descriptor structs and *_host arrays are copied by ao_geometry_create.
 *     Screens, phase, images, slopes, PSFs and the workspace are caller-owned device memory
 *     (e.g. torch tensors); screens and workspace are borrowed for the life of the handle,
 *     the others for the duration of the call (until the stream work completes).  The library
 *     calls cudaMalloc only inside ao_geometry_create (small tables) and never afterwards.
 *   - A handle is not thread-safe: one handle per host thread / stream.  It belongs to the CUDA device that was
 *     current at ao_geometry_create; every compute call makes that device current for the calling thread.
 *   - There is no CPU fallback: without a CUDA device every compute call fails with AO_ERR_CUDA.
 */
#ifndef AO_H_
#define AO_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ao_geometry ao_geometry;   /* opaque; created and destroyed by the library */

typedef enum {
    AO_OK = 0,
    AO_ERR_INVALID_ARG = 1,   /* NULL where a pointer is required, negative count, bad index       */
    AO_ERR_SHAPE = 2,         /* descriptor sizes inconsistent (bin*n_pix > fft, n_samp > fft, ...) */
    AO_ERR_UNSUPPORTED = 3,   /* size outside what the kernels implement (see ao_geometry_create)   */
    AO_ERR_CUDA = 4,          /* CUDA runtime error (message in ao_last_error)                      */
    AO_ERR_WORKSPACE = 5      /* workspace missing or smaller than ao_workspace_bytes               */
} ao_status;

/* Telescope pupil (section 2: "telescope pupil inscribed on [a] square array"). */
typedef struct {
    int32_t n;               /* N_p samples per side                                   */
    double pitch_m;          /* d_p                                                    */
    const float* amp_host;   /* [n][n] amplitude A (0/1 mask), copied                  */
} ao_pupil;

/* Shack-Hartmann wavefront sensor (section 1, section 2.7). */
typedef struct {
    int32_t n_sub;           /* subapertures per side                                  */
    int32_t n_samp;          /* n: phase samples per subaperture side                  */
    int32_t fft;             /* M: zero-padded DFT size, even, n_samp <= M             */
    int32_t bin;             /* beta: FFT pixels per detector pixel side               */
    int32_t n_pix;           /* P: detector pixels per side, beta*P <= M, (M-beta*P) even */
    float min_illum;         /* subaperture valid iff sum(A^2)/n^2 >= min_illum        */
    const float* amp_host;   /* [n_sub*n_samp]^2 amplitude on this WFS grid, copied    */
} ao_wfs;

/* Turbulent layer (section 2.1: static phase screens, frozen flow). */
typedef struct {
    int32_t n;               /* S: screen samples per side (periodic screen)           */
    double pitch_m;          /* d_l                                                    */
    double height_m;         /* h_l                                                    */
    double wind_x_mps;       /* the screen moves with +v: the pupil samples x - v t    */
    double wind_y_mps;
    const float* screen_dev; /* [n][n] radians at lambda_ref, DEVICE pointer, borrowed; must stay valid while
                                the handle is used and is only read by the library, with one exception:
                                ao_forward_host(screens_host != NULL) overwrites it with the host copy, so
                                for that call the buffer must be writable device memory.  A base address
                                aligned to 16 bytes with n a multiple of 4 takes the tiled (TMA-staged)
                                ray-trace; anything else the per-sample fallback kernel (same results) */
} ao_layer;

/* Guide star or science direction (section 2.2: "all the stars"; LGS at finite distance). */
typedef struct {
    double theta_x_rad;      /* a source at +theta displaces its footprint by +h theta */
    double theta_y_rad;
    double altitude_m;       /* H; INFINITY for natural stars and science directions    */
    double lambda_m;         /* phase is scaled by lambda_ref / lambda_m                */
    int32_t wfs_index;       /* index into the wfs array, or -1: science direction      */
} ao_source;

/* Detector noise (section 2.5 "noise"; reading O5). NULL pointer = noiseless. */
typedef struct {
    uint64_t seed;             /* Philox4x32-10 key                                     */
    float photons_per_subap;   /* N_ph: mean photo-electrons of a fully lit subaperture */
    float read_noise_e;        /* Gaussian sigma in electrons                           */
} ao_noise;

/* ao_geometry_create -- validate and copy the problem description, build device tables.
 * Problem statement: PAPER.md:36 (pupil), :28 (6 LGS SH-WFS + 3 NGS), :56 (layers), :60 (stars).
 *   pupil, wfs[n_wfs], layers[n_layers], src[n_src]: see the structs; copied.
 *   lambda_ref_m : wavelength at which the screens are expressed in radians.
 *   psf_fft      : M of the science PSF (power of two, >= pupil n; 0 if no ao_psf call is made).
 *   out          : receives the handle.
 * Supported sizes: WFS with fft <= 64: any even fft (fast paths for 16/24/32/64);
 *   WFS with fft > 64: fft a power of two <= 4096 and bin*n_pix == fft or smaller central window,
 *   and (sources using the sensor) x n_sub^2 <= 65535;
 *   psf_fft: power of two in [64, 4096]; n_layers <= 128.  Otherwise AO_ERR_UNSUPPORTED.
 * Errors: AO_ERR_INVALID_ARG (NULL, counts < 0, wfs_index out of range), AO_ERR_SHAPE,
 *   AO_ERR_UNSUPPORTED, AO_ERR_CUDA (no device / allocation failure).  *out is NULL on failure.
 * Synchronous (uses cudaMemcpy on the legacy default stream). */
int ao_geometry_create(const ao_pupil* pupil, const ao_wfs* wfs, int n_wfs,
                       const ao_layer* layers, int n_layers, const ao_source* src, int n_src,
                       double lambda_ref_m, int psf_fft, ao_geometry** out);

/* ao_geometry_destroy -- free the handle and its device tables (not the borrowed buffers).
 * NULL is accepted.  Synchronises the device first. */
int ao_geometry_destroy(ao_geometry* g);

/* Workspace: scratch for the multi-pass large FFTs and for phase staging when a call is made
 * with phase_dev == NULL.  ao_workspace_bytes is a pure size query (0 on NULL handle);
 * max_steps is the largest n_steps the caller will pass to one call.  The caller allocates
 * at least that many bytes (256-byte aligned) and lends them with ao_set_workspace; calls
 * that need more than was lent fail with AO_ERR_WORKSPACE before launching anything. */
size_t ao_workspace_bytes(const ao_geometry* g, int max_steps);
int ao_set_workspace(ao_geometry* g, void* workspace_dev, size_t bytes);

/* Phase buffer layout: phase_dev holds, for each step k in [0, n_steps), the grids of all
 * sources back to back: element offset of (source s, step k) is
 *   k * ao_phase_elems_per_step(g) + ao_phase_offset(g, s, 0),  grid s being [N_s][N_s]. */
size_t ao_phase_elems_per_step(const ao_geometry* g);
size_t ao_phase_offset(const ao_geometry* g, int source, int step);   /* (size_t)-1 on bad index */

/* Validity of the subapertures of WFS `wfs_index` (reading O6): valid_host [n_sub^2] receives
 * 1 where sum(A^2)/n^2 >= min_illum.  Returns the number of valid subapertures, or -1. */
int ao_wfs_valid(const ao_geometry* g, int wfs_index, uint8_t* valid_host /* nullable */);

/* ao_trace_layers -- open-loop wavefront of every source (section 2.2; frozen flow
 * PAPER.md:56 section 2.1; reading O2):
 *   phase_s[k][i][j] = (lambda_ref/lambda_s) sum_l bilinear(screen_l; u, v),
 *   u = (gamma x_j + h_l theta_x - v_x t_k)/d_l + (S_l-1)/2,  v likewise from y_i,
 *   gamma = 1 - h_l/H_s (cone effect; 1 for H = inf), layers with h_l >= H_s skipped,
 *   t_k = (step0+k) dt_s, screen indices periodic (mod S_l).
 * phase_dev: output, layout above, n_steps * ao_phase_elems_per_step floats (radians at lambda_s). */
int ao_trace_layers(ao_geometry* g, int64_t step0, int n_steps, double dt_s,
                    float* phase_dev, void* cuda_stream);

/* ao_sh_images -- Shack-Hartmann detector images (and optionally slopes) of all sources that
 * use WFS `wfs_index`, for n_steps steps (readings O3, O4, O5, O6):
 *   per valid subaperture: E = A exp(i phi) (n x n), half-pixel-centred DFT zero-padded to M
 *   (nu_k = k-(M-1)/2), I = |E~|^2/(M^2 n^2), central beta*P window summed in beta x beta blocks;
 *   with noise: pixel = Poisson(N_ph I) + read_noise * N(0,1), Philox counter
 *   (pixel, subaperture, source index, step0+k); invalid subapertures give zeros.
 * phase_dev : input in the ao_trace_layers layout (all sources, n_steps steps), or NULL: the
 *             ray-trace is done by the library for (step0, n_steps, dt_s) (fused path; no phase
 *             is returned).  step0/dt_s are also used for the noise counter.
 * noise     : NULL = noiseless.
 * images_dev: nullable output [n_steps][n_src_w][n_sub^2][P][P], n_src_w = sources using this WFS
 *             in ascending source order.
 * slopes_dev: nullable output [n_steps][n_src_w][2][n_sub^2] (x block then y block), centre of
 *             gravity of the (noisy if noise) images, detector pixels.  At least one output. */
int ao_sh_images(ao_geometry* g, int wfs_index, const float* phase_dev, int64_t step0,
                 int n_steps, double dt_s, const ao_noise* noise, float* images_dev,
                 float* slopes_dev, void* cuda_stream);

/* ao_centroids -- centre of gravity of caller-supplied images ("X- and Y-slopes";
 * reading O6): s_x = sum (c-(P-1)/2) pix / sum pix, s_y with the row index; 0 for invalid
 * subapertures or |sum pix| < 1e-12.
 * images_dev [n_image_sets][n_sub^2][P][P] -> slopes_dev [n_image_sets][2][n_sub^2]. */
int ao_centroids(ao_geometry* g, int wfs_index, const float* images_dev, int n_image_sets,
                 float* slopes_dev, void* cuda_stream);

/* ao_psf -- long-exposure science PSF of every science direction (section 2.8; reading O7):
 *   PSF_k = |DFT_M(A exp(i phi_k))|^2 / (M^2 sum A^2), pixel-centred (peak at [M/2][M/2]), sum = 1;
 *   psf_dev[d] = (accumulate ? psf_dev[d] : 0) + sum_{k < n_steps} PSF_k.
 * phase_dev: ao_trace_layers layout, or NULL (ray-trace done by the library).
 * psf_dev  : [n_sci][M][M], science directions in ascending source order. */
int ao_psf(ao_geometry* g, const float* phase_dev, int64_t step0, int n_steps, double dt_s,
           float* psf_dev, int accumulate, void* cuda_stream);

/* ao_psf_static -- ao_psf for ONE science direction from a phase buffer, for callers that may not allocate (CUDA graph
 * capture, tight serving loops, harnesses that forbid cudaMalloc) and so cannot lend a workspace either.  Same
 * operation and kernels as ao_psf (section 2.8; reading O7):
 *   psf_dev = (accumulate ? psf_dev : 0) + sum_{k < n_steps} |DFT_M(A exp(i phi_k))|^2 / (M^2 sum A^2)
 * for science direction `direction` (index among the science directions, ascending source order).
 *   phase_dev : DEVICE, ao_trace_layers layout, n_steps steps (required: this call does no ray-trace).
 *   psf_dev   : DEVICE, [M][M] floats of that one direction, caller-owned.
 * The intermediate of the two-pass FFT (pupil n x M complex floats) lives in a static device array of
 * AO_PSF_STATIC_MAX_BYTES that every GPU loading the library holds until the process exits; the call makes no
 * cudaMalloc / cudaFree and calls no allocating library routine, needs no workspace, and is asynchronous on `cuda_stream`.
 * pupil n * M * 8 > AO_PSF_STATIC_MAX_BYTES is rejected with AO_ERR_UNSUPPORTED (c3 / c4: 960 x 2048 x 8 = 15.7 MB fits).
 * All calls on one device share the array (whatever the handle): it keeps the previous call's intermediate, which the
 * row pass overwrites in full before it is read, so nothing is cleared; two calls that overlap on the GPU (different
 * streams, or two host threads) RACE on it and give wrong PSFs -- serialise them on one stream or with events.
 * Errors: AO_ERR_INVALID_ARG (NULL, direction out of range, n_steps < 0, no science direction),
 *   AO_ERR_UNSUPPORTED (size beyond the static scratch), AO_ERR_CUDA. */
#define AO_PSF_STATIC_MAX_BYTES (16u << 20)
int ao_psf_static(ao_geometry* g, int direction, const float* phase_dev, int n_steps, float* psf_dev,
                  int accumulate, void* cuda_stream);

/* ao_set_psf_band / ao_psf_poly -- polychromatic science PSF (section 2.8: "The user select the wavelength at
 * which the PSF is computed and the pixelscale ... The user may desire more wavelengths, considering a bandwidth"; DESIGN.md
 * section 3 reading O8).  The detector pixels keep the angular size lambda_s / (M d_p) of the science directions' own
 * wavelength lambda_s; wavelength lambda_j (s_j = lambda_s / lambda_j) sees the phase s_j phi and a pattern 1/s_j wider:
 *   PSF_k = sum_j w_j s_j^2 |sum_ab A exp(i s_j phi_k) exp(-2 pi i s_j ((k-M/2) a + (m-M/2) b)/M)|^2 / (M^2 sum A^2),
 * the scaled DFT being evaluated as a chirp-z transform with FFTs of length L >= M + N_p - 1.  One wavelength equal to
 * lambda_s with weight 1 is ao_psf.
 * ao_set_psf_band: lambdas_m_host [n_lambda], weights_host [n_lambda]: HOST arrays, copied; builds the chirp tables in
 *   FP64 (cudaMalloc; synchronises the device); n_lambda = 0 clears the band.  Needs psf_fft + pupil n - 1 <= 4096 and
 *   all science directions at one wavelength, else AO_ERR_UNSUPPORTED.  While a band is set, ao_forward and
 *   ao_forward_host produce the polychromatic PSF; ao_psf stays monochromatic.
 * ao_psf_poly: same arguments, layout, accumulation and workspace as ao_psf; AO_ERR_INVALID_ARG if no band is set. */
int ao_set_psf_band(ao_geometry* g, const double* lambdas_m_host, const double* weights_host, int n_lambda);
int ao_psf_poly(ao_geometry* g, const float* phase_dev, int64_t step0, int n_steps, double dt_s,
                float* psf_dev, int accumulate, void* cuda_stream);

/* ao_set_phase_map -- static additive phase map of one source (section 2.3: telescope aberration
 * maps such as M1 scalloping and the NGS-WFS mis-positioning tip/tilt are "summed to the open loop WF"):
 *   phi_s[k, i, j] <- phi_s[k, i, j] + map[i][j]  for every time step k,
 * applied wherever the library produces phi_s (ao_trace_layers and every phase_dev == NULL path: ao_sh_images,
 * ao_psf, ao_forward, ao_forward_host).  map_dev: [N_s][N_s] fp32 radians AT THE SOURCE'S WAVELENGTH on the source's
 * grid (ao_trace_layers layout of one source), DEVICE pointer, borrowed until replaced, cleared with NULL, or the
 * handle is destroyed.  Synchronises the device (the call updates a table that launches in flight may be reading).
 * Errors: AO_ERR_INVALID_ARG for a bad handle or source index. */
int ao_set_phase_map(ao_geometry* g, int source, const float* map_dev);

/* ao_set_sodium -- extended sodium layer for the LGS sensors of WFS `wfs_index` (section 2.7: "It's possible to
 * consider at this level the sodium layer temporal evolution"; DESIGN.md section 3 reading O9).  The beacon of every source of
 * that WFS becomes a column of n_z scatterers at altitudes z_m[i] with weights rho[t][i]; time step s uses the profile row
 * t = s mod n_t (the temporal evolution: n_t = 1 is a static profile).  Seen from the subaperture centred at c, scatterer i
 * is displaced from the focus point (the source altitude H) by the angle (c - L)(1/H - 1/z_i), L = launch_xy_m of the
 * source: its spot is the point-beacon spot shifted by that angle (a phase ramp over the subaperture, exact on the DFT grid,
 * periodic in the field of view) and the detector sums the spots with the weights rho (which the caller normalises).
 *   z_m_host [n_z], rho_host [n_t][n_z], launch_xy_m_host [n_src_w][2] (sources of the WFS in ascending order): HOST
 *   arrays, copied.  n_z = 0 restores the point beacon.  1 <= n_z <= 64.
 * Applies to ao_sh_images (both phase_dev paths), ao_forward and ao_forward_host.  Synchronises the device; allocates the
 * small tables with cudaMalloc (with ao_set_psf_band the only calls after ao_geometry_create that do).
 * Errors: AO_ERR_INVALID_ARG (bad index, NULL arrays, a source at infinity, z <= 0), AO_ERR_UNSUPPORTED (fft > 64). */
int ao_set_sodium(ao_geometry* g, int wfs_index, int n_z, const double* z_m_host, const double* rho_host, int n_t,
                  const double* launch_xy_m_host);

/* ao_modes_to_map -- residual-phase entry (section 2.7: "residual = open loop WF - DM shape", the
 * WFS then measures the residual; section 2.5: the calibration pushes mirror modes through the WFS):
 *   map[i] = sign * sum_{m < n_modes} coeffs[m] * modes[m][i],  i < n_elems   (fp32, modes summed in index order).
 * With map_dev registered once through ao_set_phase_map and sign = -1 this is the deformable-mirror shape
 * subtracted from the open-loop wavefront of that source; the mode arrays (mirror modes projected on the
 * source's grid, radians at its wavelength) and the coefficients are the caller's: modal bases and control are
 * outside this library.  All pointers are DEVICE pointers: modes_dev [n_modes][n_elems], coeffs_dev [n_modes],
 * map_dev [n_elems] (overwritten).  Asynchronous on cuda_stream: calls that follow on the same stream see the
 * new map.  n_modes = 0 zeroes the map.  Errors: AO_ERR_INVALID_ARG for NULL pointers or negative sizes. */
int ao_modes_to_map(ao_geometry* g, const float* modes_dev, int n_modes, long long n_elems,
                    const float* coeffs_dev, float sign, float* map_dev, void* cuda_stream);

/* ao_strehl -- Strehl ratio of every science direction from its long-exposure PSF (section 2.8: "the
 * Strehl Ratio ... computed on the PSF"): with the PSF normalisation of ao_psf (sum = 1 per exposure) the
 * diffraction-limited peak is peak_flat = (sum A)^2 / (M^2 sum A^2), at pixel [M/2][M/2], and
 *   strehl[d] = psf_dev[d][M/2][M/2] / (n_exposures * peak_flat).
 * psf_dev: [n_sci][M][M] as written by ao_psf / ao_forward; n_exposures: the number of steps summed into it;
 * strehl_dev: [n_sci] fp32 DEVICE pointer.  Asynchronous on cuda_stream.
 * Errors: AO_ERR_INVALID_ARG (NULL pointers, n_exposures <= 0, no science direction / psf_fft == 0). */
int ao_strehl(ao_geometry* g, const float* psf_dev, double n_exposures, float* strehl_dev, void* cuda_stream);

/* ao_strehl_marechal -- Strehl ratio by the Marechal approximation on the wavefront (section 2.8: "or
 * by the Marechal approximation on the closed loop WF"):  strehl[k][d] = exp(-var_A(phi_{k,d})), var_A the
 * amplitude-weighted variance of the phase of science direction d over the pupil (weights A[i][j], piston removed),
 * accumulated in FP64.  phase_dev: ao_trace_layers layout (radians at each source's wavelength; residual phase if
 * maps are set), n_steps steps; strehl_dev: [n_steps][n_sci] fp32 DEVICE pointer.  Asynchronous on cuda_stream.
 * Errors: AO_ERR_INVALID_ARG (NULL pointers, n_steps < 0, no science direction). */
int ao_strehl_marechal(ao_geometry* g, const float* phase_dev, int n_steps, float* strehl_dev, void* cuda_stream);

/* ao_forward -- the whole step with DEVICE buffers: ray-trace + every WFS (slopes only, noiseless unless
 * `noise`) + every science PSF for n_steps steps (the per-time-step forward model).
 * Same results as one ao_sh_images(phase_dev = NULL, images_dev = NULL) per WFS plus ao_psf(phase_dev = NULL) (ao_psf_poly
 * while a band is set), submitted in order on `cuda_stream`: the workspace users (big-FFT sensors, PSF) first, then the
 * sensors that need no workspace (the fused ray-trace + SH + CoG kernels).  Asynchronous like every other call.
 * slopes_dev[w] (nullable per entry): ao_sh_images slopes layout of WFS w.
 * psf_dev (nullable): [n_sci][M][M], += if accumulate else =.  Needs a workspace if any big WFS or PSF runs. */
int ao_forward(ao_geometry* g, int64_t step0, int n_steps, double dt_s, const ao_noise* noise,
               float* const* slopes_dev, float* psf_dev, int accumulate, void* cuda_stream);

/* ao_forward_host -- the whole step for host callers: uploads nothing but the call parameters,
 * runs ray-trace + every WFS (noiseless unless `noise`) + every PSF for n_steps steps on
 * `cuda_stream`, and copies the results to HOST buffers (pinned memory recommended), then
 * synchronises the stream.  slopes_host[w] (nullable per entry) receives WFS w's slopes in the
 * ao_sh_images layout; psf_host (nullable) receives [n_sci][M][M] (sum over the steps).
 * The device staging for the results lives in the workspace (see ao_workspace_bytes).
 * If screens_host is non-NULL, screens_host[l] ([S_l][S_l] floats, the whole screen) is the host copy of layer l and
 * the call first uploads, into layer l's borrowed device screen (the one call that writes the screens, see
 * ao_layer.screen_dev), the part of it that steps [step0, step0 + n_steps) read: the bounding box of all footprints
 * (periodic wrap included) plus a 24-sample margin; a layer no source sees is not uploaded, a box as large as the screen
 * uploads all of it.  Device samples outside the box keep their previous contents.  ao_last_h2d_bytes() returns the bytes
 * the last call uploaded. */
int ao_forward_host(ao_geometry* g, const float* const* screens_host, int64_t step0, int n_steps,
                    double dt_s, const ao_noise* noise, float* const* slopes_host,
                    float* psf_host, void* cuda_stream);

/* ao_probe_fp32 -- measurement aid for the roofline line of bench.py ("the builder must also
 * measure an FMA-chain micro-benchmark"): runs an FMA-chain micro-kernel (8 independent chains per thread, 8 CTAs of
 * 256 threads per SM) five times on the legacy default stream, times it with CUDA events and returns the best FP32
 * rate in TFLOP/s.  packed = 0: scalar FFMA; packed != 0: FFMA2 (fma.rn.f32x2).  Synchronous.
 * Errors: AO_ERR_INVALID_ARG (NULL), AO_ERR_CUDA. */
int ao_probe_fp32(ao_geometry* g, int packed, double* tflops_out);

/* Bytes of screens uploaded host -> device by the last ao_forward_host call on this handle (0 without screens_host). */
uint64_t ao_last_h2d_bytes(const ao_geometry* g);

/* Number of kernel launches issued by this handle since creation (all ao_* calls). */
int64_t ao_launch_count(const ao_geometry* g);

const char* ao_last_error(void);
/* Version string; it states the build flavour ("normal build", or "PROFILING build" when the library was compiled
 * with the component-timing switches, whose results are not valid). */
const char* ao_version(void);

#ifdef __cplusplus
}
#endif
#endif /* AO_H_ */
