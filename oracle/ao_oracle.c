/* ao_oracle.c -- FP64 CPU oracle for the per-time-step optical forward model.
 *
 * TEST INFRASTRUCTURE ONLY.  This file is the parity oracle and the timed CPU
 * baseline.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, load or call it.  It shares no code, header,
 * table or helper with the CUDA path (paper_1608_00386_b200/csrc) and neither
 * includes the other.
 *
 * The paper (arxiv 1608.00386, /root/reference/PAPER.md) names the operations but
 * gives no formula; every definition below is the reading fixed in SURVEY.md §8(c)
 * (O1..O7), restated in DESIGN.md §3.  Each function cites the passage it follows.
 * Everything is the plain definition written out: finite sums in double precision,
 * a direct separable DFT for FFT sizes <= 64 and a textbook iterative radix-2 FFT
 * (pinned against the direct DFT by tests/test_oracle_pins.py) for the large
 * power-of-two sizes.  OpenMP only distributes independent outputs over threads.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): brute-force O(N^4) DFT, numpy FFT,
 * Dirichlet-kernel closed forms and the tilt/CoG table of SURVEY.md §8(c)
 * (tests/golden/), Parseval, flat->zero slopes, piston invariance, linear-screen
 * bilinear exactness, integer/half-pixel shifts, cone scaling, periodicity,
 * cuRAND's host Philox4_32_10 generator, scipy.stats.poisson.ppf (mu up to 1e4), Poisson/Gauss statistics.
 * O8 (polychromatic PSF, oracle/__init__.py psf_poly) and O9 (LGS elongation, aoref_sh_images_elong) are pinned by
 * closed forms too (one wavelength = aoref_psf, the 2M crop identity, Dirichlet products; delta profile = aoref_sh_images,
 * whole-pixel shifts along the launch-to-subaperture direction, energy).  No function here is "parity unpinned".
 *
 * Layout: all arrays row-major [y][x], x fastest.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define AOREF_OK 0
#define AOREF_ERR_ARG 1
#define AOREF_ERR_ALLOC 2

#ifndef M_PI
#define M_PI 3.14159265358979323846
#endif

int aoref_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void aoref_set_num_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

static inline int64_t pmod(int64_t a, int64_t m)
{
    int64_t r = a % m;
    return r < 0 ? r + m : r;
}

/* ------------------------------------------------------------------------------------
 * O2  Ray-trace (§2.1 frozen flow; §2.2 open-loop wavefront for
 * all stars and the geometrical projection of a finite-distance LGS).
 *
 * phase[i][j] = (lambda_ref/lambda) * sum_l bilinear(screen_l; u, v)
 *   x_j = (j-(N-1)/2) d,  y_i likewise                         (O1 grid)
 *   gamma = 1 - h_l/H (1 for H = inf); layers with h_l >= H are skipped
 *   X = gamma x_j + h_l theta_x - v_x t ;  u = X/d_l + (S-1)/2 ;  same for Y, v
 *   j0 = floor(u), fx = u-j0, i0 = floor(v), fy = v-i0, indices taken mod S (periodic)
 *   value = (1-fy)[(1-fx) s00 + fx s01] + fy[(1-fx) s10 + fx s11]
 * One source, one time t per call.
 */
int aoref_trace(int n_layers, const float* const* screens, const int32_t* S,
                const double* pitch_m, const double* height_m,
                const double* wind_x, const double* wind_y,
                double theta_x, double theta_y, double altitude_m,
                double lambda_m, double lambda_ref_m,
                int N, double d, double t, double* phase)
{
    if (n_layers < 0 || N <= 0 || !phase) return AOREF_ERR_ARG;
    #pragma omp parallel for schedule(static)
    for (int i = 0; i < N; ++i) {
        const double y = ((double)i - (double)(N - 1) / 2.0) * d;
        for (int j = 0; j < N; ++j) {
            const double x = ((double)j - (double)(N - 1) / 2.0) * d;
            double acc = 0.0;
            for (int l = 0; l < n_layers; ++l) {
                const double h = height_m[l];
                if (!(h < altitude_m)) continue;
                const double gamma = isinf(altitude_m) ? 1.0 : 1.0 - h / altitude_m;
                const double X = gamma * x + h * theta_x - wind_x[l] * t;
                const double Y = gamma * y + h * theta_y - wind_y[l] * t;
                const int64_t Sl = S[l];
                const double u = X / pitch_m[l] + (double)(Sl - 1) / 2.0;
                const double v = Y / pitch_m[l] + (double)(Sl - 1) / 2.0;
                const double fu = floor(u), fv = floor(v);
                const double fx = u - fu, fy = v - fv;
                const int64_t j0 = pmod((int64_t)fu, Sl), j1 = pmod((int64_t)fu + 1, Sl);
                const int64_t i0 = pmod((int64_t)fv, Sl), i1 = pmod((int64_t)fv + 1, Sl);
                const float* s = screens[l];
                const double s00 = s[i0 * Sl + j0], s01 = s[i0 * Sl + j1];
                const double s10 = s[i1 * Sl + j0], s11 = s[i1 * Sl + j1];
                acc += (1.0 - fy) * ((1.0 - fx) * s00 + fx * s01)
                     + fy * ((1.0 - fx) * s10 + fx * s11);
            }
            phase[(size_t)i * N + j] = acc * (lambda_ref_m / lambda_m);
        }
    }
    return AOREF_OK;
}

/* ------------------------------------------------------------------------------------
 * Textbook iterative radix-2 decimation-in-time FFT, forward sign exp(-2 pi i k a / M),
 * in place on M complex values with the given stride.  M must be a power of two.
 * Used only for M > 64 ("for M = 1024 and 2048, an iterative radix-2
 * FFT (own code), checked against the direct DFT").
 */
static void fft_radix2(double* re, double* im, int M, size_t stride, const double* tw_re,
                       const double* tw_im)
{
    /* bit reversal */
    for (int i = 1, j = 0; i < M; ++i) {
        int bit = M >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) {
            double tr = re[i * stride]; re[i * stride] = re[j * stride]; re[j * stride] = tr;
            double ti = im[i * stride]; im[i * stride] = im[j * stride]; im[j * stride] = ti;
        }
    }
    for (int len = 2; len <= M; len <<= 1) {
        const int half = len >> 1, step = M / len;
        for (int base = 0; base < M; base += len) {
            for (int k = 0; k < half; ++k) {
                const double wr = tw_re[k * step], wi = tw_im[k * step];  /* exp(-2 pi i k/len) */
                const size_t a = (size_t)(base + k) * stride, b = (size_t)(base + k + half) * stride;
                const double xr = re[b] * wr - im[b] * wi, xi = re[b] * wi + im[b] * wr;
                re[b] = re[a] - xr; im[b] = im[a] - xi;
                re[a] += xr;        im[a] += xi;
            }
        }
    }
}

static int is_pow2(int M) { return M > 0 && (M & (M - 1)) == 0; }

/* ------------------------------------------------------------------------------------
 * O3 / O7  Centred 2-D DFT of an n x n block zero-padded to M x M (
 * PAPER.md:28,82 name the Shack-Hartmann sensor, PAPER.md:86 the PSF module).
 *
 *   out[k][m] = sum_{a<n} sum_{b<n} in[a][b] exp(-2 pi i (nu_k a + nu_m b)/M)
 *   half_pixel = 1:  nu_k = k - (M-1)/2   (Shack-Hartmann: spot on a 4-pixel junction)
 *   half_pixel = 0:  nu_k = k - M/2       (PSF: peak on pixel [M/2][M/2])
 *   method 0: direct separable DFT, FP64 twiddle table W[q] = exp(-i pi q / M), q mod 2M
 *             (rows then columns; the plain definition, any even or odd M)
 *   method 1: pre-multiply by exp(+2 pi i c (a+b)/M) with c = (M-1)/2 or M/2, then the
 *             radix-2 FFT over rows and columns (M power of two)
 * out_re/out_im: [M][M].  threads: OpenMP inside (rows / columns are independent).
 */
int aoref_cdft2(const double* in_re, const double* in_im, int n, int M, int half_pixel,
                int method, double* out_re, double* out_im)
{
    if (n <= 0 || M < n || !in_re || !in_im || !out_re || !out_im) return AOREF_ERR_ARG;
    if (method == 1 && !is_pow2(M)) return AOREF_ERR_ARG;
    const int twoM = 2 * M;
    double* W_re = (double*)malloc(sizeof(double) * twoM);
    double* W_im = (double*)malloc(sizeof(double) * twoM);
    if (!W_re || !W_im) { free(W_re); free(W_im); return AOREF_ERR_ALLOC; }
    for (int q = 0; q < twoM; ++q) {          /* W[q] = exp(-i pi q / M) */
        W_re[q] = cos(M_PI * (double)q / (double)M);
        W_im[q] = -sin(M_PI * (double)q / (double)M);
    }
    /* twice the centre: nu_k = k - c2/2 */
    const int c2 = half_pixel ? (M - 1) : M;

    if (method == 0) {
        /* rows: R[a][m] = sum_b in[a][b] W[((2m - c2) b) mod 2M] */
        double* R_re = (double*)malloc(sizeof(double) * (size_t)n * M);
        double* R_im = (double*)malloc(sizeof(double) * (size_t)n * M);
        if (!R_re || !R_im) { free(R_re); free(R_im); free(W_re); free(W_im); return AOREF_ERR_ALLOC; }
        #pragma omp parallel for schedule(static) if (M > 64)
        for (int a = 0; a < n; ++a)
            for (int m = 0; m < M; ++m) {
                double sr = 0.0, si = 0.0;
                for (int b = 0; b < n; ++b) {
                    const int q = (int)pmod((int64_t)(2 * m - c2) * b, twoM);
                    const double xr = in_re[a * n + b], xi = in_im[a * n + b];
                    sr += xr * W_re[q] - xi * W_im[q];
                    si += xr * W_im[q] + xi * W_re[q];
                }
                R_re[(size_t)a * M + m] = sr; R_im[(size_t)a * M + m] = si;
            }
        /* columns: out[k][m] = sum_a R[a][m] W[((2k - c2) a) mod 2M] */
        #pragma omp parallel for schedule(static) if (M > 64)
        for (int k = 0; k < M; ++k)
            for (int m = 0; m < M; ++m) {
                double sr = 0.0, si = 0.0;
                for (int a = 0; a < n; ++a) {
                    const int q = (int)pmod((int64_t)(2 * k - c2) * a, twoM);
                    const double xr = R_re[(size_t)a * M + m], xi = R_im[(size_t)a * M + m];
                    sr += xr * W_re[q] - xi * W_im[q];
                    si += xr * W_im[q] + xi * W_re[q];
                }
                out_re[(size_t)k * M + m] = sr; out_im[(size_t)k * M + m] = si;
            }
        free(R_re); free(R_im);
    } else {
        /* exp(-2 pi i (k - c2/2) a / M) = exp(-2 pi i k a/M) * exp(+i pi c2 a / M) = ... * conj(W[(c2 a) mod 2M]) */
        double* tw_re = (double*)malloc(sizeof(double) * (M / 2 + 1));
        double* tw_im = (double*)malloc(sizeof(double) * (M / 2 + 1));
        if (!tw_re || !tw_im) { free(tw_re); free(tw_im); free(W_re); free(W_im); return AOREF_ERR_ALLOC; }
        for (int k = 0; k < M / 2 + 1; ++k) {     /* exp(-2 pi i k / M) */
            tw_re[k] = cos(2.0 * M_PI * (double)k / (double)M);
            tw_im[k] = -sin(2.0 * M_PI * (double)k / (double)M);
        }
        memset(out_re, 0, sizeof(double) * (size_t)M * M);
        memset(out_im, 0, sizeof(double) * (size_t)M * M);
        for (int a = 0; a < n; ++a)
            for (int b = 0; b < n; ++b) {
                const int q = (int)pmod((int64_t)c2 * (a + b), twoM);
                const double pr = W_re[q], pi = -W_im[q];         /* conj(W[q]) */
                const double xr = in_re[a * n + b], xi = in_im[a * n + b];
                out_re[(size_t)a * M + b] = xr * pr - xi * pi;
                out_im[(size_t)a * M + b] = xr * pi + xi * pr;
            }
        #pragma omp parallel for schedule(static)
        for (int a = 0; a < n; ++a)                 /* rows a >= n are zero and stay zero */
            fft_radix2(out_re + (size_t)a * M, out_im + (size_t)a * M, M, 1, tw_re, tw_im);
        #pragma omp parallel for schedule(static)
        for (int m = 0; m < M; ++m)
            fft_radix2(out_re + m, out_im + m, M, (size_t)M, tw_re, tw_im);
        free(tw_re); free(tw_im);
    }
    free(W_re); free(W_im);
    return AOREF_OK;
}

/* ------------------------------------------------------------------------------------
 * O3 + O4  Shack-Hartmann detector images ("Shack-Hartmann Wavefront Sensors",
 * PAPER.md:82 "WFS modules compute the vector signals"; SURVEY.md §8(c) O3, O4, O6 validity).
 *
 * Per subaperture (p, q) of an n_sub x n_sub grid with n x n samples each:
 *   illum = sum A^2 / n^2 ; valid = illum >= min_illum ; invalid -> image = 0
 *   E[a][b] = A exp(i phi) on the block ; Etilde = half-pixel-centred DFT, zero-padded to M
 *   I[k][m] = |Etilde|^2 / (M^2 n^2)
 *   pix[r][c] = sum of I over k in [k0+beta r, k0+beta r+beta), m likewise, k0 = (M-beta P)/2
 * phase, amp: [n_sub*n][n_sub*n]; images: [n_sub*n_sub][P][P]; valid: [n_sub*n_sub].
 */
int aoref_sh_images(const double* phase, const float* amp, int n_sub, int n, int M, int beta,
                    int P, double min_illum, double* images, uint8_t* valid)
{
    if (!phase || !amp || !images || !valid || n_sub <= 0 || n <= 0 || M < n || beta <= 0 ||
        P <= 0 || beta * P > M || ((M - beta * P) & 1))
        return AOREF_ERR_ARG;
    const int N = n_sub * n, nsa = n_sub * n_sub, big = (M > 64);
    if (big && !is_pow2(M)) return AOREF_ERR_ARG;
    const int k0 = (M - beta * P) / 2;
    int err = 0;
    #pragma omp parallel for schedule(dynamic, 4) if (!big)
    for (int sa = 0; sa < nsa; ++sa) {
        const int p = sa / n_sub, q = sa % n_sub;
        double* img = images + (size_t)sa * P * P;
        for (int i = 0; i < P * P; ++i) img[i] = 0.0;
        double illum = 0.0;
        for (int a = 0; a < n; ++a)
            for (int b = 0; b < n; ++b) {
                const double A = amp[(size_t)(p * n + a) * N + q * n + b];
                illum += A * A;
            }
        illum /= (double)n * n;
        valid[sa] = (uint8_t)(illum >= min_illum);
        if (!valid[sa]) continue;
        double* e_re = (double*)malloc(sizeof(double) * n * n);
        double* e_im = (double*)malloc(sizeof(double) * n * n);
        double* o_re = (double*)malloc(sizeof(double) * (size_t)M * M);
        double* o_im = (double*)malloc(sizeof(double) * (size_t)M * M);
        if (!e_re || !e_im || !o_re || !o_im) {
            free(e_re); free(e_im); free(o_re); free(o_im);
            #pragma omp atomic write
            err = AOREF_ERR_ALLOC;
            continue;
        }
        for (int a = 0; a < n; ++a)
            for (int b = 0; b < n; ++b) {
                const size_t g = (size_t)(p * n + a) * N + q * n + b;
                const double A = amp[g], ph = phase[g];
                e_re[a * n + b] = A * cos(ph);
                e_im[a * n + b] = A * sin(ph);
            }
        aoref_cdft2(e_re, e_im, n, M, 1, big ? 1 : 0, o_re, o_im);
        const double norm = 1.0 / ((double)M * M * (double)n * n);
        for (int r = 0; r < P; ++r)
            for (int c = 0; c < P; ++c) {
                double s = 0.0;
                for (int k = k0 + beta * r; k < k0 + beta * r + beta; ++k)
                    for (int m = k0 + beta * c; m < k0 + beta * c + beta; ++m) {
                        const double xr = o_re[(size_t)k * M + m], xi = o_im[(size_t)k * M + m];
                        s += (xr * xr + xi * xi) * norm;
                    }
                img[r * P + c] = s;
            }
        free(e_re); free(e_im); free(o_re); free(o_im);
    }
    return err;
}

/* ------------------------------------------------------------------------------------
 * O9  Shack-Hartmann images of a laser guide star with an extended sodium layer (section 2.7: "It's possible
 * to consider at this level the sodium layer temporal evolution"; DESIGN.md section 3
 * reading O9).  The paper gives no formula; the reading is plain geometry.
 *
 * The beacon is a column of n_z scatterers at altitudes z_i with weights rho_i (the sodium profile at this time step,
 * caller-supplied), on the line from the launch point L = (launch_x, launch_y) [m, pupil plane] to the focus point at
 * altitude H.  Seen from the subaperture centred at c, the scatterer at z_i is displaced from the focus point by the angle
 *     delta_i = (c - L) (1/H - 1/z_i)                                (small angles; zero for z_i = H)
 * which is a tilt of  alpha_i = 2 pi delta_i d / lambda  radians per sample across the subaperture (d = sample pitch),
 * i.e. a shift of the spot by delta_i M d / lambda FFT pixels along c - L.  The detector integrates incoherently:
 *     I = sum_i rho_i |DFT_M( A exp(i (phi + alpha_ix b + alpha_iy a)) )|^2 / (M^2 n^2),   then binned as in O4.
 * Subaperture centre: x_c = ((q n + (n-1)/2) - (N-1)/2) d, y_c with p (O1 grid).  Validity as in aoref_sh_images.
 * n_z = 1 with z_0 = H reproduces aoref_sh_images.
 */
int aoref_sh_images_elong(const double* phase, const float* amp, int n_sub, int n, int M, int beta, int P,
                          double min_illum, double d, double lambda_m, double H, double launch_x, double launch_y,
                          int n_z, const double* z, const double* rho, double* images, uint8_t* valid)
{
    if (!phase || !amp || !images || !valid || !z || !rho || n_z <= 0 || n_sub <= 0 || n <= 0 || M < n || beta <= 0 ||
        P <= 0 || beta * P > M || ((M - beta * P) & 1) || M > 64)
        return AOREF_ERR_ARG;
    const int N = n_sub * n, nsa = n_sub * n_sub;
    const int k0 = (M - beta * P) / 2;
    int err = 0;
    #pragma omp parallel for schedule(dynamic, 4)
    for (int sa = 0; sa < nsa; ++sa) {
        const int p = sa / n_sub, q = sa % n_sub;
        double* img = images + (size_t)sa * P * P;
        for (int i = 0; i < P * P; ++i) img[i] = 0.0;
        double illum = 0.0;
        for (int a = 0; a < n; ++a)
            for (int b = 0; b < n; ++b) {
                const double A = amp[(size_t)(p * n + a) * N + q * n + b];
                illum += A * A;
            }
        illum /= (double)n * n;
        valid[sa] = (uint8_t)(illum >= min_illum);
        if (!valid[sa]) continue;
        double* e_re = (double*)malloc(sizeof(double) * n * n);
        double* e_im = (double*)malloc(sizeof(double) * n * n);
        double* o_re = (double*)malloc(sizeof(double) * (size_t)M * M);
        double* o_im = (double*)malloc(sizeof(double) * (size_t)M * M);
        if (!e_re || !e_im || !o_re || !o_im) {
            free(e_re); free(e_im); free(o_re); free(o_im);
            #pragma omp atomic write
            err = AOREF_ERR_ALLOC;
            continue;
        }
        const double xc = (((double)q * n + (double)(n - 1) / 2.0) - (double)(N - 1) / 2.0) * d;
        const double yc = (((double)p * n + (double)(n - 1) / 2.0) - (double)(N - 1) / 2.0) * d;
        const double norm = 1.0 / ((double)M * M * (double)n * n);
        for (int iz = 0; iz < n_z; ++iz) {
            const double g = 2.0 * M_PI * (1.0 / H - 1.0 / z[iz]) * d / lambda_m;       /* rad per sample per metre of baseline */
            const double ax = g * (xc - launch_x), ay = g * (yc - launch_y);
            for (int a = 0; a < n; ++a)
                for (int b = 0; b < n; ++b) {
                    const size_t gi = (size_t)(p * n + a) * N + q * n + b;
                    const double A = amp[gi], ph = phase[gi] + ax * (double)b + ay * (double)a;
                    e_re[a * n + b] = A * cos(ph);
                    e_im[a * n + b] = A * sin(ph);
                }
            aoref_cdft2(e_re, e_im, n, M, 1, 0, o_re, o_im);
            for (int r = 0; r < P; ++r)
                for (int c = 0; c < P; ++c) {
                    double s = 0.0;
                    for (int k = k0 + beta * r; k < k0 + beta * r + beta; ++k)
                        for (int m = k0 + beta * c; m < k0 + beta * c + beta; ++m) {
                            const double xr = o_re[(size_t)k * M + m], xi = o_im[(size_t)k * M + m];
                            s += (xr * xr + xi * xi) * norm;
                        }
                    img[r * P + c] += rho[iz] * s;
                }
        }
        free(e_re); free(e_im); free(o_re); free(o_im);
    }
    return err;
}

/* ------------------------------------------------------------------------------------
 * O6  Centre of gravity ("X- and Y-slopes").
 *   sx = sum_{r,c} (c-(P-1)/2) pix / sum pix ;  sy with r ; detector pixels, +x = +column.
 *   valid[i] == 0 (if given) or |sum pix| < 1e-12  ->  sx = sy = 0.
 * images: [n_img][P][P]; sx, sy: [n_img].
 */
int aoref_centroids(const double* images, int n_img, int P, const uint8_t* valid,
                    double* sx, double* sy)
{
    if (!images || !sx || !sy || n_img < 0 || P <= 0) return AOREF_ERR_ARG;
    #pragma omp parallel for schedule(static)
    for (int i = 0; i < n_img; ++i) {
        const double* img = images + (size_t)i * P * P;
        double s = 0.0, mx = 0.0, my = 0.0;
        for (int r = 0; r < P; ++r)
            for (int c = 0; c < P; ++c) {
                const double v = img[r * P + c];
                s += v;
                mx += ((double)c - (double)(P - 1) / 2.0) * v;
                my += ((double)r - (double)(P - 1) / 2.0) * v;
            }
        if ((valid && !valid[i]) || fabs(s) < 1e-12) { sx[i] = 0.0; sy[i] = 0.0; }
        else { sx[i] = mx / s; sy[i] = my / s; }
    }
    return AOREF_OK;
}

/* ------------------------------------------------------------------------------------
 * O7  Science PSF (§2.8).
 *   PSF = |DFT_M(A exp(i phi))|^2 / (M^2 sum A^2), pixel-centred (nu_k = k - M/2), so that
 *   sum PSF = 1 and a flat pupil peaks at [M/2][M/2] with value (sum A)^2/(M^2 sum A^2).
 *   accumulate != 0: psf += PSF (long exposure is the running sum).
 * phase, amp: [N][N]; psf: [M][M].  M <= 64: direct DFT; else radix-2 FFT (power of two).
 */
int aoref_psf(const double* phase, const float* amp, int N, int M, int accumulate, double* psf)
{
    if (!phase || !amp || !psf || N <= 0 || M < N) return AOREF_ERR_ARG;
    if (M > 64 && !is_pow2(M)) return AOREF_ERR_ARG;
    double* e_re = (double*)malloc(sizeof(double) * (size_t)N * N);
    double* e_im = (double*)malloc(sizeof(double) * (size_t)N * N);
    double* o_re = (double*)malloc(sizeof(double) * (size_t)M * M);
    double* o_im = (double*)malloc(sizeof(double) * (size_t)M * M);
    if (!e_re || !e_im || !o_re || !o_im) { free(e_re); free(e_im); free(o_re); free(o_im); return AOREF_ERR_ALLOC; }
    double sumA2 = 0.0;
    for (size_t g = 0; g < (size_t)N * N; ++g) {
        const double A = amp[g];
        sumA2 += A * A;
        e_re[g] = A * cos(phase[g]);
        e_im[g] = A * sin(phase[g]);
    }
    int rc = aoref_cdft2(e_re, e_im, N, M, 0, M > 64 ? 1 : 0, o_re, o_im);
    if (rc == AOREF_OK) {
        const double norm = sumA2 > 0.0 ? 1.0 / ((double)M * M * sumA2) : 0.0;
        #pragma omp parallel for schedule(static)
        for (int k = 0; k < M; ++k)
            for (int m = 0; m < M; ++m) {
                const size_t g = (size_t)k * M + m;
                const double v = (o_re[g] * o_re[g] + o_im[g] * o_im[g]) * norm;
                psf[g] = accumulate ? psf[g] + v : v;
            }
    }
    free(e_re); free(e_im); free(o_re); free(o_im);
    return rc;
}

/* ------------------------------------------------------------------------------------
 * O5  Detector noise ("possible environment conditions (noise)"; BASELINE.json c2
 * "Poisson+Gaussian(3 e-) detector noise from seed").
 *
 * Philox4x32-10 (Salmon et al., SC'11: the published counter-based generator, restated):
 * ten rounds of
 *   hi0,lo0 = M0 * c0 ; hi1,lo1 = M1 * c2
 *   c = (hi1 ^ c1 ^ k0, lo1, hi0 ^ c3 ^ k1, lo0) ; key += (W0, W1) between rounds
 */
void aoref_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
    for (int r = 0; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)M0 * c0, p1 = (uint64_t)M1 * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        const uint32_t n1 = (uint32_t)p1;
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        const uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += W0; k1 += W1;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* u = ((w >> 8) + 0.5) 2^-24 : in (0,1), exactly representable in fp32 and fp64. */
static inline double u24(uint32_t w) { return ((double)(w >> 8) + 0.5) * (1.0 / 16777216.0); }

/* Poisson by inversion of the CDF on u: the smallest k with u <= F(k; mu), F(k) = sum_{j<=k} e^-mu mu^j / j!.
 *   mu < 64: sequential search from 0: k = 0; p = c = exp(-mu); while u > c: k++, p *= mu/k, c += p.
 *   mu >= 64 (reading O5 as revised in round 2: exp(-mu) underflows FP64 above mu ~ 745 and the
 *   search from 0 then returns floor(mu)+1 for every u): the same inverse CDF, searched from the mode m = floor(mu):
 *     p_m = exp(m ln mu - mu - lgamma(m+1));  F(m) = p_m + p_{m-1} + ... (p_{j-1} = p_j j/mu, until a term adds nothing);
 *     u <= F(m): walk down while u <= F(k) - p_k (then k--), else walk up while u > F(k) (k++, p *= mu/k, F += p).
 * Pinned against scipy.stats.poisson.ppf for mu up to 1e4 and by the variance at mu = 800, 1e3, 1e4. */
static int32_t poisson_inv(double mu, double u)
{
    if (!(mu > 0.0)) return 0;
    if (mu < 64.0) {
        int32_t k = 0;
        double p = exp(-mu), c = p;
        while (u > c && k < 100000) {
            ++k;
            p *= mu / (double)k;
            c += p;
            if (p == 0.0 && (double)k > mu) break;   /* CDF saturated below u by rounding */
        }
        return k;
    }
    const double m = floor(mu);
    const double pm = exp(m * log(mu) - mu - lgamma(m + 1.0));
    double Fm = pm, p = pm;
    for (double j = m; j >= 1.0; j -= 1.0) {          /* F(m): terms below the mode, largest first */
        p *= j / mu;
        const double next = Fm + p;
        if (next == Fm) break;
        Fm = next;
    }
    double k = m, c = Fm;
    p = pm;
    if (u <= c) {
        while (k > 0.0 && u <= c - p) { c -= p; p *= k / mu; k -= 1.0; }
    } else {
        while (u > c && k < 2147483000.0) {
            k += 1.0;
            p *= mu / k;
            c += p;
            if (p == 0.0) break;                      /* CDF saturated below u by rounding */
        }
    }
    return (int32_t)k;
}

/*   mu = photons * I ; key = (seed lo, seed hi) ; counter = (pixel-in-image, subaperture, source, step)
 *   w0..w3 = Philox ; k = Poisson^-1(mu; u(w0)) ; z = sqrt(-2 ln u(w1)) cos(2 pi u(w2))
 *   out = k + read_noise * z.   Invalid subapertures stay 0.  counts (nullable) receives k.
 * images/out: [n_img][P][P]  (normalised noiseless images in, electrons out).
 */
int aoref_noise(const double* images, int n_img, int P, const uint8_t* valid, uint64_t seed,
                uint32_t source, uint32_t step, double photons, double read_noise,
                double* out, int32_t* counts)
{
    if (!images || !out || n_img < 0 || P <= 0) return AOREF_ERR_ARG;
    const uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    #pragma omp parallel for schedule(static)
    for (int sa = 0; sa < n_img; ++sa)
        for (int px = 0; px < P * P; ++px) {
            const size_t g = (size_t)sa * P * P + px;
            if (valid && !valid[sa]) { out[g] = 0.0; if (counts) counts[g] = 0; continue; }
            const uint32_t ctr[4] = { (uint32_t)px, (uint32_t)sa, source, step };
            uint32_t w[4];
            aoref_philox4x32_10(ctr, key, w);
            const double mu = photons * images[g];
            const int32_t k = poisson_inv(mu, u24(w[0]));
            const double z = sqrt(-2.0 * log(u24(w[1]))) * cos(2.0 * M_PI * u24(w[2]));
            out[g] = (double)k + read_noise * z;
            if (counts) counts[g] = k;
        }
    return AOREF_OK;
}
