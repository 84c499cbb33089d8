"""ctypes binding and step driver for the FP64 CPU oracle (oracle/ao_oracle.c).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs.  Never imported by paper_1608_00386_b200.
It takes the plain descriptors of paper_1608_00386_b200.inputs (which hold no
arithmetic of the method) but imports nothing from the CUDA path.
"""
from __future__ import annotations

import ctypes as C
import math
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ao_oracle.c")
_LIB = os.path.join(_HERE, "libao_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp oracle/ao_oracle.c -> oracle/libao_oracle.so (in tree)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra",
               "-fno-fast-math", _SRC, "-o", _LIB, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


_dp = C.POINTER(C.c_double)
_fp = C.POINTER(C.c_float)
_u8p = C.POINTER(C.c_uint8)
_i32p = C.POINTER(C.c_int32)
_u32p = C.POINTER(C.c_uint32)


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        L.aoref_num_threads.restype = C.c_int
        L.aoref_set_num_threads.argtypes = [C.c_int]
        L.aoref_trace.argtypes = [C.c_int, C.POINTER(_fp), _i32p, _dp, _dp, _dp, _dp,
                                  C.c_double, C.c_double, C.c_double, C.c_double, C.c_double,
                                  C.c_int, C.c_double, C.c_double, _dp]
        L.aoref_cdft2.argtypes = [_dp, _dp, C.c_int, C.c_int, C.c_int, C.c_int, _dp, _dp]
        L.aoref_sh_images.argtypes = [_dp, _fp, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int,
                                      C.c_double, _dp, _u8p]
        L.aoref_sh_images_elong.argtypes = [_dp, _fp, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_double,
                                            C.c_double, C.c_double, C.c_double, C.c_double, C.c_double,
                                            C.c_int, _dp, _dp, _dp, _u8p]
        L.aoref_centroids.argtypes = [_dp, C.c_int, C.c_int, _u8p, _dp, _dp]
        L.aoref_psf.argtypes = [_dp, _fp, C.c_int, C.c_int, C.c_int, _dp]
        L.aoref_philox4x32_10.argtypes = [_u32p, _u32p, _u32p]
        L.aoref_philox4x32_10.restype = None
        L.aoref_noise.argtypes = [_dp, C.c_int, C.c_int, _u8p, C.c_uint64, C.c_uint32, C.c_uint32,
                                  C.c_double, C.c_double, _dp, _i32p]
        _lib = L
    return _lib


def _d(a):
    return a.ctypes.data_as(_dp)


def _check(rc, what):
    if rc != 0:
        raise RuntimeError(f"oracle {what} failed with status {rc}")


def num_threads() -> int:
    return int(lib().aoref_num_threads())


def set_num_threads(n: int) -> None:
    lib().aoref_set_num_threads(int(n))


# ------------------------------------------------------------------------------- O2
def trace(layers, theta_x, theta_y, altitude_m, lambda_m, lambda_ref_m, N, d, t) -> np.ndarray:
    """phase[N][N] (fp64 radians at lambda_m) for one source at time t.  `layers`: inputs.Layer list."""
    nl = len(layers)
    scr = [np.ascontiguousarray(l.screen, dtype=np.float32) for l in layers]
    ptrs = (_fp * max(nl, 1))(*[s.ctypes.data_as(_fp) for s in scr])
    S = np.array([l.n for l in layers], dtype=np.int32)
    pitch = np.array([l.pitch_m for l in layers], dtype=np.float64)
    h = np.array([l.height_m for l in layers], dtype=np.float64)
    wx = np.array([l.wind_x_mps for l in layers], dtype=np.float64)
    wy = np.array([l.wind_y_mps for l in layers], dtype=np.float64)
    out = np.empty((N, N), dtype=np.float64)
    _check(lib().aoref_trace(nl, ptrs, S.ctypes.data_as(_i32p), _d(pitch), _d(h), _d(wx), _d(wy),
                             float(theta_x), float(theta_y), float(altitude_m), float(lambda_m),
                             float(lambda_ref_m), int(N), float(d), float(t), _d(out)), "trace")
    return out


# ------------------------------------------------------------------------------- O3
def cdft2(block: np.ndarray, M: int, half_pixel: bool, method: int) -> np.ndarray:
    """Centred DFT of a complex n x n block zero-padded to M x M (see aoref_cdft2)."""
    n = block.shape[0]
    re = np.ascontiguousarray(block.real, dtype=np.float64)
    im = np.ascontiguousarray(block.imag, dtype=np.float64)
    o_re = np.empty((M, M)); o_im = np.empty((M, M))
    _check(lib().aoref_cdft2(_d(re), _d(im), n, M, int(half_pixel), int(method), _d(o_re), _d(o_im)),
           "cdft2")
    return o_re + 1j * o_im


# ------------------------------------------------------------------------------- O3+O4
def sh_images(phase: np.ndarray, amp: np.ndarray, n_sub, n, M, beta, P, min_illum):
    """-> images [n_sub^2][P][P] fp64, valid [n_sub^2] uint8."""
    phase = np.ascontiguousarray(phase, dtype=np.float64)
    amp = np.ascontiguousarray(amp, dtype=np.float32)
    assert phase.shape == (n_sub * n, n_sub * n) and amp.shape == phase.shape
    img = np.empty((n_sub * n_sub, P, P), dtype=np.float64)
    valid = np.empty(n_sub * n_sub, dtype=np.uint8)
    _check(lib().aoref_sh_images(_d(phase), amp.ctypes.data_as(_fp), n_sub, n, M, beta, P,
                                 float(min_illum), _d(img), valid.ctypes.data_as(_u8p)), "sh_images")
    return img, valid


# ------------------------------------------------------------------------------- O9
def sh_images_elong(phase, amp, n_sub, n, M, beta, P, min_illum, d, lambda_m, H, launch_xy, z, rho):
    """LGS images with an extended sodium layer (aoref_sh_images_elong): z, rho = altitudes [m] and weights of the
    scatterers, launch_xy = launch point [m].  -> images [n_sub^2][P][P] fp64, valid [n_sub^2] uint8."""
    phase = np.ascontiguousarray(phase, dtype=np.float64)
    amp = np.ascontiguousarray(amp, dtype=np.float32)
    z = np.ascontiguousarray(z, dtype=np.float64); rho = np.ascontiguousarray(rho, dtype=np.float64)
    assert phase.shape == (n_sub * n, n_sub * n) and amp.shape == phase.shape and z.shape == rho.shape
    img = np.empty((n_sub * n_sub, P, P), dtype=np.float64)
    valid = np.empty(n_sub * n_sub, dtype=np.uint8)
    _check(lib().aoref_sh_images_elong(_d(phase), amp.ctypes.data_as(_fp), n_sub, n, M, beta, P, float(min_illum),
                                       float(d), float(lambda_m), float(H), float(launch_xy[0]), float(launch_xy[1]),
                                       int(z.size), _d(z), _d(rho), _d(img), valid.ctypes.data_as(_u8p)),
           "sh_images_elong")
    return img, valid


# ------------------------------------------------------------------------------- O6
def centroids(images: np.ndarray, valid=None):
    """images [n][P][P] -> slopes [2][n] (x block then y block), detector pixels."""
    images = np.ascontiguousarray(images, dtype=np.float64)
    n_img, P = images.shape[0], images.shape[-1]
    out = np.empty((2, n_img), dtype=np.float64)
    vp = None
    if valid is not None:
        valid = np.ascontiguousarray(valid, dtype=np.uint8)
        vp = valid.ctypes.data_as(_u8p)
    _check(lib().aoref_centroids(_d(images), n_img, P, vp, _d(out[0]), _d(out[1])), "centroids")
    return out


# ------------------------------------------------------------------------------- O7
def psf(phase: np.ndarray, amp: np.ndarray, M: int, into: np.ndarray | None = None) -> np.ndarray:
    phase = np.ascontiguousarray(phase, dtype=np.float64)
    amp = np.ascontiguousarray(amp, dtype=np.float32)
    N = phase.shape[0]
    acc = 1
    if into is None:
        into = np.zeros((M, M), dtype=np.float64)
        acc = 0
    _check(lib().aoref_psf(_d(phase), amp.ctypes.data_as(_fp), N, M, acc, _d(into)), "psf")
    return into


# ------------------------------------------------------------------------------- O8
def psf_poly(phase: np.ndarray, amp: np.ndarray, M: int, lambda_s: float, lambdas, weights,
             into: np.ndarray | None = None) -> np.ndarray:
    """Polychromatic science PSF on the detector pixel grid of the direction's own wavelength lambda_s (PAPER.md:86
    section 2.8: "The user select the wavelength at which the PSF is computed and the pixelscale ... The user may desire
    more wavelengths, considering a bandwidth"; DESIGN.md section 3 reading O8).  phase is in radians at lambda_s.
    With s_j = lambda_s / lambda_j (the same optical path is s_j phi radians at lambda_j, and the diffraction pattern
    is 1/s_j times wider on pixels of fixed angular size lambda_s / (M d_p)):
        E_j = A exp(i s_j phi);   Et_j[k][m] = sum_ab E_j[a][b] exp(-2 pi i s_j ((k - M/2) a + (m - M/2) b) / M)
        PSF = sum_j w_j s_j^2 |Et_j|^2 / (M^2 sum A^2)
    (s_j^2: flux per pixel of fixed solid angle; every wavelength integrates to w_j over the whole plane).  One
    wavelength equal to lambda_s with weight 1 is aoref_psf.  The definition written out: the scaled DFT is two dense
    FP64 matrix products F E F^T with F[k][a] = exp(-2 pi i s_j (k - M/2) a / M) (numpy matmul is the library step)."""
    ph = np.asarray(phase, dtype=np.float64)
    A = np.asarray(amp, dtype=np.float64)
    N = ph.shape[0]
    out = np.zeros((M, M), dtype=np.float64) if into is None else into
    sumA2 = float((A * A).sum())
    kap = np.arange(M, dtype=np.float64) - M / 2.0
    a = np.arange(N, dtype=np.float64)
    for lam, w in zip(lambdas, weights):
        s = float(lambda_s) / float(lam)
        E = A * np.exp(1j * s * ph)
        F = np.exp(-2j * np.pi * s * np.outer(kap, a) / M)               # [M][N]
        Et = (F @ E) @ F.T
        out += float(w) * s * s * (Et.real ** 2 + Et.imag ** 2) / (M * M * sumA2)
    return out


# ------------------------------------------------------------------------------- O5
def philox4x32_10(ctr, key) -> np.ndarray:
    c = np.asarray(ctr, dtype=np.uint32).copy(); k = np.asarray(key, dtype=np.uint32).copy()
    o = np.empty(4, dtype=np.uint32)
    lib().aoref_philox4x32_10(c.ctypes.data_as(_u32p), k.ctypes.data_as(_u32p), o.ctypes.data_as(_u32p))
    return o


def noise(images: np.ndarray, valid, seed: int, source: int, step: int, photons: float,
          read_noise: float):
    """-> (noisy images [n][P][P] in electrons, Poisson counts int32 [n][P][P])."""
    images = np.ascontiguousarray(images, dtype=np.float64)
    n_img, P = images.shape[0], images.shape[-1]
    out = np.empty_like(images); counts = np.empty(images.shape, dtype=np.int32)
    vp = None
    if valid is not None:
        valid = np.ascontiguousarray(valid, dtype=np.uint8)
        vp = valid.ctypes.data_as(_u8p)
    _check(lib().aoref_noise(_d(images), n_img, P, vp, C.c_uint64(seed & (2 ** 64 - 1)),
                             C.c_uint32(source & 0xFFFFFFFF), C.c_uint32(step & 0xFFFFFFFF),
                             float(photons), float(read_noise), _d(out),
                             counts.ctypes.data_as(_i32p)), "noise")
    return out, counts


# ------------------------------------------------------------------------------- step driver
def strehl(psf_sum: np.ndarray, amp: np.ndarray, n_exposures: float) -> float:
    """Strehl ratio on the PSF (section 2.8): peak pixel [M/2][M/2] of the long exposure over n_exposures times
    the diffraction-limited peak (sum A)^2 / (M^2 sum A^2) of the PSF normalisation of reading O7.  FP64."""
    M = psf_sum.shape[0]
    a = np.asarray(amp, dtype=np.float64)
    peak_flat = a.sum() ** 2 / (M * M * (a * a).sum())
    return float(psf_sum[M // 2, M // 2] / (n_exposures * peak_flat))


def strehl_marechal(phase: np.ndarray, amp: np.ndarray) -> float:
    """Marechal approximation (section 2.8): exp(-var_A(phi)), the amplitude-weighted phase variance over
    the pupil with the weighted mean (piston) removed.  FP64, the definition written out."""
    w = np.asarray(amp, dtype=np.float64)
    p = np.asarray(phase, dtype=np.float64)
    mean = (w * p).sum() / w.sum()
    return float(np.exp(-(w * (p - mean) ** 2).sum() / w.sum()))


def modes_to_map(modes: np.ndarray, coeffs: np.ndarray, sign: float) -> np.ndarray:
    """Residual-phase entry (PAPER.md:82 section 2.7, :74 section 2.5): map = sign * sum_m coeffs[m] modes[m], FP64.
    The plain definition: one numpy contraction over the mode index."""
    m = np.asarray(modes, dtype=np.float64)
    c = np.asarray(coeffs, dtype=np.float64)
    return float(sign) * np.tensordot(c, m, axes=(0, 0))


def forward(cfg, step0: int = 0, n_steps: int = 1, *, want_phase=True, want_wfs=True,
            want_psf=True, noise_on=False, sources=None):
    """Run the whole forward model of `cfg` (inputs.Config) for steps step0..step0+n_steps-1.

    Returns a dict:
      phase[s]   : list over steps of [N_s][N_s] fp64          (if want_phase)
      images[s]  : [n_steps][n_sub^2][P][P]   (WFS sources; noiseless, normalised)
      noisy[s], counts[s] : as images, electrons / Poisson counts   (if noise_on and cfg.noise)
      slopes[s]  : [n_steps][2][n_sub^2]      (from noisy images if noise_on else noiseless)
      valid[w]   : [n_sub^2] uint8 per WFS
      psf[s]     : [M][M] long-exposure SUM over the steps (science sources)
    cfg.phase_maps[s] (optional, [N_s][N_s] radians at the source's wavelength) is added to the traced phase of
    source s at every step (section 2.3) before the WFS and the PSF see it.
    cfg.sodium (optional, inputs.Sodium): the sensors of that WFS see an extended beacon (reading O9); time step
    step0 + k uses profile row (step0 + k) mod n_t.  cfg.psf_band (optional, (wavelengths, weights)): the science PSF
    is the polychromatic sum of reading O8 on the pixel grid of each direction's own wavelength.
    Plain loop over steps and sources; every number comes from ao_oracle.c (the map sum is one numpy add).
    """
    res = {"phase": {}, "images": {}, "noisy": {}, "counts": {}, "slopes": {}, "valid": {}, "psf": {}}
    srcs = range(len(cfg.sources)) if sources is None else sources
    for s in srcs:
        src = cfg.sources[s]
        N = cfg.grid_n(s)
        d = cfg.grid_pitch(s)
        w = src.wfs_index
        if w >= 0 and not want_wfs and not want_phase:
            continue
        if w < 0 and not want_psf and not want_phase:
            continue
        ph_list, im_list, sl_list, nz_list, ct_list = [], [], [], [], []
        acc = None
        for k in range(n_steps):
            t = (step0 + k) * cfg.dt_s
            ph = trace(cfg.layers, src.theta_x_rad, src.theta_y_rad, src.altitude_m, src.lambda_m,
                       cfg.lambda_ref_m, N, d, t)
            pm = getattr(cfg, "phase_maps", {}).get(s)
            if pm is not None:      # static aberration map summed to the open-loop wavefront (section 2.3)
                ph = ph + np.asarray(pm, dtype=np.float64)
            if want_phase:
                ph_list.append(ph)
            if w >= 0 and want_wfs:
                W = cfg.wfs[w]
                na = getattr(cfg, "sodium", None)
                if na is not None and na.wfs_index == w:
                    rho = np.asarray(na.rho, dtype=np.float64)
                    img, valid = sh_images_elong(ph, W.amp, W.n_sub, W.n_samp, W.fft, W.bin, W.n_pix, W.min_illum,
                                                 d, src.lambda_m, src.altitude_m,
                                                 na.launch_xy_m[cfg.sources_of_wfs(w).index(s)], na.z_m,
                                                 rho[(step0 + k) % rho.shape[0]])
                else:
                    img, valid = sh_images(ph, W.amp, W.n_sub, W.n_samp, W.fft, W.bin, W.n_pix, W.min_illum)
                res["valid"][w] = valid
                im_list.append(img)
                use = img
                if noise_on and cfg.noise is not None:
                    nz, ct = noise(img, valid, cfg.noise.seed, s, step0 + k,
                                   cfg.noise.photons_per_subap, cfg.noise.read_noise_e)
                    nz_list.append(nz); ct_list.append(ct)
                    use = nz
                sl_list.append(centroids(use, valid))
            if w < 0 and want_psf and cfg.psf_fft:
                band = getattr(cfg, "psf_band", None)
                if band is not None:
                    acc = psf_poly(ph, cfg.pupil.amp, cfg.psf_fft, src.lambda_m, band[0], band[1], into=acc)
                elif acc is None:
                    acc = psf(ph, cfg.pupil.amp, cfg.psf_fft)
                else:
                    psf(ph, cfg.pupil.amp, cfg.psf_fft, into=acc)
        if want_phase:
            res["phase"][s] = ph_list
        if im_list:
            res["images"][s] = np.stack(im_list)
            res["slopes"][s] = np.stack(sl_list)
        if nz_list:
            res["noisy"][s] = np.stack(nz_list)
            res["counts"][s] = np.stack(ct_list)
        if acc is not None:
            res["psf"][s] = acc
    return res
