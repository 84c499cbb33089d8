"""Seeded synthetic inputs and plain descriptors for the optical forward model.

This module serves BOTH the CUDA path and the FP64 oracle and therefore holds
none of the method's arithmetic (no ray-trace, no DFT, no centroid): only
  * descriptor dataclasses (pupil, WFS, layer, source, noise, config),
  * the binary pupil masks (geometry evaluated in FP64),
  * the seeded von Karman phase-screen generator (§2.1: screens
    "computed by DFT ... Kolmogorov or Von Karman models"; harness, not hot path),
  * the five BASELINE.json workloads c0..c4 and reduced copies of them.

It imports neither `oracle/` nor the CUDA binding.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field, replace
from typing import List, Optional

import numpy as np

ARCSEC = math.pi / 180.0 / 3600.0
LAMBDA_REF = 500e-9          # wavelength at which r0 is quoted and screens are in radians
R0_REF = 0.157               # m at 500 nm (BASELINE.json configs)
L0_REF = 25.0                # m outer scale
SEED_BASE = 160800386        # PCG64(seed = 160800386 + config_index)


# --------------------------------------------------------------------------- descriptors
@dataclass
class Pupil:
    n: int                   # samples per side (N_p)
    pitch_m: float           # d_p
    r_out_m: float
    r_in_m: float
    amp: Optional[np.ndarray] = None   # [n][n] float32 0/1 mask


@dataclass
class WFS:
    n_sub: int               # subapertures per side
    n_samp: int              # samples per subaperture side (n)
    fft: int                 # M
    bin: int                 # beta
    n_pix: int               # P  (bin*n_pix <= fft)
    min_illum: float = 0.5
    amp: Optional[np.ndarray] = None   # [n_sub*n_samp]^2 float32 mask on this WFS grid

    @property
    def n_grid(self) -> int:
        return self.n_sub * self.n_samp


@dataclass
class Layer:
    n: int                   # screen side S
    pitch_m: float           # d_l
    height_m: float          # h_l
    wind_x_mps: float
    wind_y_mps: float
    weight: float            # Cn2 fraction (used by the generator only)
    screen: Optional[np.ndarray] = None   # [n][n] float32 radians at LAMBDA_REF (host copy)
    screen_dev: Optional[object] = None   # the same screen as a torch CUDA tensor (keep_on_device)


@dataclass
class Source:
    theta_x_rad: float
    theta_y_rad: float
    altitude_m: float        # math.inf for NGS / science
    lambda_m: float
    wfs_index: int           # -1: science direction on the pupil grid


@dataclass
class Noise:
    seed: int
    photons_per_subap: float
    read_noise_e: float


@dataclass
class Sodium:
    """Extended sodium layer seen by the LGS sensors of one WFS (reading O9): scatterer altitudes z [n_z],
    weights rho [n_t][n_z] (row (step mod n_t) is the profile of a time step: the temporal evolution), and the launch
    point of every source of that WFS [n_src_w][2] in metres in the pupil plane."""
    wfs_index: int
    z_m: np.ndarray
    rho: np.ndarray
    launch_xy_m: np.ndarray


@dataclass
class Config:
    name: str
    pupil: Pupil
    wfs: List[WFS]
    layers: List[Layer]
    sources: List[Source]
    n_steps: int
    dt_s: float = 2e-3
    lambda_ref_m: float = LAMBDA_REF
    psf_fft: int = 0         # M of the science PSF (0: no science PSF)
    noise: Optional[Noise] = None
    seed: int = SEED_BASE
    r0_m: float = R0_REF
    L0_m: float = L0_REF
    notes: dict = field(default_factory=dict)
    # static additive phase maps: source index -> [N_s][N_s] float32 radians at the source's wavelength
    phase_maps: dict = field(default_factory=dict)
    sodium: Optional[Sodium] = None          # NEXT-3: LGS spot elongation (None: point beacon at the source altitude)
    psf_band: Optional[tuple] = None         # NEXT-4: (wavelengths_m [n], weights [n]) of the polychromatic science PSF

    # ---- derived shapes (no arithmetic of the method; only sizes) ----
    def grid_n(self, s: int) -> int:
        w = self.sources[s].wfs_index
        return self.pupil.n if w < 0 else self.wfs[w].n_grid

    def grid_pitch(self, s: int) -> float:
        """d_s = N_p d_p / N_s: every grid spans the pupil width."""
        return self.pupil.n * self.pupil.pitch_m / self.grid_n(s)

    def sources_of_wfs(self, w: int) -> List[int]:
        return [i for i, s in enumerate(self.sources) if s.wfs_index == w]

    def science_sources(self) -> List[int]:
        return [i for i, s in enumerate(self.sources) if s.wfs_index < 0]

    def phase_elems_per_step(self) -> int:
        return sum(self.grid_n(s) ** 2 for s in range(len(self.sources)))


# --------------------------------------------------------------------------- masks
def annulus_mask(n: int, pitch_m: float, r_out_m: float, r_in_m: float) -> np.ndarray:
    """amp[i][j] = 1 if r_in^2 <= x_j^2 + y_i^2 <= r_out^2, x_j = (j-(n-1)/2) pitch (FP64)."""
    x = (np.arange(n, dtype=np.float64) - (n - 1) / 2.0) * pitch_m
    r2 = x[None, :] ** 2 + x[:, None] ** 2
    return ((r2 <= r_out_m * r_out_m) & (r2 >= r_in_m * r_in_m)).astype(np.float32)


def fill_masks(cfg: Config) -> Config:
    p = cfg.pupil
    p.amp = annulus_mask(p.n, p.pitch_m, p.r_out_m, p.r_in_m)
    width = p.n * p.pitch_m
    for w in cfg.wfs:
        w.amp = annulus_mask(w.n_grid, width / w.n_grid, p.r_out_m, p.r_in_m)
    return cfg


# --------------------------------------------------------------------------- screens
def von_karman_psd(f2: "np.ndarray", r0_m: float, L0_m: float):
    """Phi(f) = 0.0229 r0^(-5/3) (f^2 + L0^-2)^(-11/6)   [rad^2 m^2] (ref [28])."""
    return 0.0229 * r0_m ** (-5.0 / 3.0) * (f2 + L0_m ** -2.0) ** (-11.0 / 6.0)


def screen_expected_variance(n: int, pitch_m: float, r0_m: float, L0_m: float) -> float:
    """Exact expected variance of a generated screen: sum_{f != 0} Phi(f) df^2."""
    df = 1.0 / (n * pitch_m)
    fx = np.fft.fftfreq(n, d=pitch_m)
    f2 = fx[None, :] ** 2 + fx[:, None] ** 2
    psd = von_karman_psd(f2, r0_m, L0_m)
    psd[0, 0] = 0.0
    return float(psd.sum() * df * df)


def von_karman_pair(n: int, pitch_m: float, r0_m: float, L0_m: float,
                    rng: np.random.Generator, device: str = "cpu", as_torch: bool = False):
    """Two independent periodic von Karman screens [n][n] float32 (radians at 500 nm).

    c(f) = (xi1 + i xi2) sqrt(Phi(f)) df, c(0) = 0, phi = n^2 ifft2(c); Re and Im are
    independent screens.  The Gaussian numbers always come from the numpy PCG64
    stream `rng` (host); only the inverse FFT may run on `device` through
    torch.fft (used for the 8192^2 screens of c4 on the GPU box).
    """
    df = 1.0 / (n * pitch_m)
    xi = rng.standard_normal((2, n, n))
    if device == "cpu":
        fx = np.fft.fftfreq(n, d=pitch_m)
        f2 = fx[None, :] ** 2 + fx[:, None] ** 2
        amp = np.sqrt(von_karman_psd(f2, r0_m, L0_m)) * df
        amp[0, 0] = 0.0
        c = (xi[0] + 1j * xi[1]) * amp
        del xi
        phi = np.fft.ifft2(c) * float(n * n)
        return phi.real.astype(np.float32), phi.imag.astype(np.float32)
    import torch
    dev = torch.device(device)
    fx = torch.fft.fftfreq(n, d=pitch_m, dtype=torch.float64, device=dev)
    f2 = fx[None, :] ** 2 + fx[:, None] ** 2
    amp = torch.sqrt(0.0229 * r0_m ** (-5.0 / 3.0) * (f2 + L0_m ** -2.0) ** (-11.0 / 6.0)) * df
    amp[0, 0] = 0.0
    c = torch.complex(torch.from_numpy(xi[0]).to(dev), torch.from_numpy(xi[1]).to(dev)) * amp
    del xi, amp, f2
    phi = torch.fft.ifft2(c) * float(n * n)
    del c
    re = phi.real.to(torch.float32).contiguous()
    im = phi.imag.to(torch.float32).contiguous()
    del phi
    if as_torch:
        return re, im
    return re.cpu().numpy(), im.cpu().numpy()


def fill_screens(cfg: Config, device: str = "cpu", keep_on_device: bool = False) -> Config:
    """Generate one screen per layer with r0_l = r0 w_l^(-3/5): each layer carries sqrt(weight).

    keep_on_device (device must be CUDA): leave the screens as torch CUDA tensors in
    `screen_dev` (no host round trip for the 9.4 GB of c4); `screens_to_host` fetches them.
    """
    rng = np.random.default_rng(np.random.PCG64(cfg.seed + 7919))
    spare = None
    for lay in cfg.layers:
        # r0_l^(-5/3) = r0^(-5/3) w_l, so a unit-weight screen times sqrt(w_l) is layer l's screen;
        # one FFT yields a pair (Re, Im): the spare serves the next layer of the same shape
        if spare is not None and spare[0] == (lay.n, lay.pitch_m):
            unit = spare[1]
            spare = None
        else:
            unit, b = von_karman_pair(lay.n, lay.pitch_m, cfg.r0_m, cfg.L0_m, rng, device,
                                      as_torch=keep_on_device)
            spare = ((lay.n, lay.pitch_m), b)
        if keep_on_device:
            lay.screen_dev = unit * float(np.float32(math.sqrt(lay.weight)))   # fp32 tensor * python float
            lay.screen = None
        else:
            lay.screen = (unit * np.float32(math.sqrt(lay.weight))).astype(np.float32)
    return cfg


def screens_to_host(cfg: Config) -> Config:
    """Fill `screen` (numpy, host) from `screen_dev` for layers generated with keep_on_device."""
    for lay in cfg.layers:
        if lay.screen is None and lay.screen_dev is not None:
            lay.screen = lay.screen_dev.cpu().numpy()
    return cfg


# --------------------------------------------------------------------------- workloads
ELT_WEIGHTS_10 = [0.45, 0.10, 0.08, 0.07, 0.06, 0.06, 0.05, 0.05, 0.04, 0.04]   # BASELINE.json c2


def _ring(radius_arcsec: float, azimuths_deg, altitude_m, lambda_m, wfs_index):
    out = []
    for az in azimuths_deg:
        a = math.radians(az)
        out.append(Source(radius_arcsec * ARCSEC * math.cos(a), radius_arcsec * ARCSEC * math.sin(a),
                          altitude_m, lambda_m, wfs_index))
    return out


def _winds(rng: np.random.Generator, n_layers: int):
    speed = rng.uniform(5.0, 30.0, n_layers)
    direction = rng.uniform(0.0, 2.0 * math.pi, n_layers)
    return speed * np.cos(direction), speed * np.sin(direction)


def make_config(index: int, *, n_sub: Optional[int] = None, screen_n: Optional[int] = None,
                n_steps: Optional[int] = None, lgs_fft: int = 32, ngs_samp: Optional[int] = None,
                psf_fft: Optional[int] = None, n_layers: Optional[int] = None,
                with_screens: bool = True, device: str = "cpu", keep_on_device: bool = False) -> Config:
    """Build workload c<index> of BASELINE.json.

    The keyword overrides shrink a workload while keeping its recipe (same pitch, same
    samples per subaperture, same FFT/bin sizes, same source constellation): `n_sub`
    scales the pupil (N_p = n_sub * N_p_full / n_sub_full), `screen_n` the screens.
    With no overrides the full-size workload is returned.
    """
    seed = SEED_BASE + index
    rng = np.random.default_rng(np.random.PCG64(seed))
    if index == 0:
        ns = n_sub or 10
        npup = ns * 8
        pupil = Pupil(npup, 0.1, npup * 0.1 / 2.0, 0.0)
        wfs = [WFS(ns, 8, 16, 2, 8)]
        S = screen_n or 256
        layers = [Layer(S, 0.1, 0.0, 10.0, 0.0, 1.0)]
        sources = [Source(0.0, 0.0, math.inf, 589e-9, 0)]
        cfg = Config("c0_tiny_ngs_scao", pupil, wfs, layers, sources, n_steps or 1, seed=seed)
    elif index == 1:
        ns = n_sub or 80
        npup = ns * 12
        scale = ns / 80.0
        pupil = Pupil(npup, 0.04, npup * 0.04 / 2.0, 5.5 * scale)
        wfs = [WFS(ns, 12, 24, 4, 6)]
        S = screen_n or 2048
        layers = [Layer(S, 0.04, h, 10.0, 0.0, w) for h, w in
                  zip([0.0, 4000.0, 12000.0], [0.6, 0.25, 0.15])]
        sources = [Source(0.0, 0.0, math.inf, 0.8e-6, 0)]
        cfg = Config("c1_elt_ngs_scao", pupil, wfs, layers, sources, n_steps or 100, seed=seed)
    elif index in (2, 3, 4):
        ns = n_sub or 80
        npup = ns * 12                      # pupil grid: 960 at full size, pitch 0.04 m
        scale = ns / 80.0
        pupil = Pupil(npup, 0.04, npup * 0.04 / 2.0, 5.5 * scale)
        if index == 4:
            L = n_layers or 35
            heights = np.linspace(0.0, 26500.0, L)
            w = rng.uniform(0.0, 1.0, L)
            weights = (w / w.sum()).tolist()
            S = screen_n or 8192
            M = lgs_fft
        else:
            L = n_layers or 10
            heights = np.linspace(0.0, 25000.0, L)
            weights = ELT_WEIGHTS_10[:L]
            S = screen_n or 2048
            M = 32
        wx, wy = _winds(rng, L)
        layers = [Layer(S, 0.04, float(h), float(a), float(b), float(wt))
                  for h, a, b, wt in zip(heights, wx, wy, weights)]
        wfs = [WFS(ns, M // 2, M, M // 8, 8)]
        sources = _ring(45.0, [60.0 * s for s in range(6)], 90e3, 589e-9, 0)
        noise = None
        psf = 0
        steps = {2: 100, 3: 50, 4: 1000}[index]
        if index == 2:
            noise = Noise(seed=seed, photons_per_subap=1000.0, read_noise_e=3.0)
        if index in (3, 4):
            nsamp = ngs_samp or npup // 2          # 2x2 subapertures of N_p/2 samples
            Mn = 1 << (2 * nsamp - 1).bit_length()  # next power of two >= 2*nsamp (480 -> 1024)
            wfs.append(WFS(2, nsamp, Mn, 8, Mn // 8, min_illum=0.5))
            sources += _ring(80.0, [30.0, 150.0, 270.0], math.inf, 0.8e-6, 1)
            psf = psf_fft or (1 << (2 * npup - 1).bit_length())   # 960 -> 2048
            if index == 3:
                dirs = [(a, b) for b in (-30.0, 0.0, 30.0) for a in (-30.0, 0.0, 30.0)] + [(45.0, 45.0)]
            else:
                dirs = [(0.0, 0.0)]
            sources += [Source(a * ARCSEC, b * ARCSEC, math.inf, 2.2e-6, -1) for a, b in dirs]
        name = {2: "c2_maory_lgs_wfs", 3: "c3_full_mcao_step", 4: f"c4_throughput_M{M}"}[index]
        cfg = Config(name, pupil, wfs, layers, sources, n_steps or steps, psf_fft=psf,
                     noise=noise, seed=seed)
    else:
        raise ValueError("config index must be 0..4")
    fill_masks(cfg)
    if with_screens:
        fill_screens(cfg, device=device, keep_on_device=keep_on_device)
    return cfg


def sodium_profile(cfg: Config, wfs_index: int = 0, n_z: int = 5, n_t: int = 8, mean_m: float = 90e3,
                   fwhm_m: float = 10e3, launch: str = "centre", seed: Optional[int] = None) -> Sodium:
    """Synthetic sodium layer (the paper's profile is not given): n_z equally spaced scatterers over +-1.25 FWHM
    around a mean altitude that drifts by up to +-500 m over the n_t time samples, Gaussian weights plus a seeded
    sporadic component on one slab, each row normalised to 1.  launch = "centre" (behind the secondary mirror) or
    "side" (at the pupil edge, on the azimuth of each beacon).  Input data only: no arithmetic of the method."""
    rng = np.random.default_rng(np.random.PCG64((cfg.seed if seed is None else seed) + 4099))
    sigma = fwhm_m / 2.3548200450309493
    z = mean_m + np.linspace(-1.25, 1.25, n_z) * fwhm_m
    drift = 500.0 * np.sin(2.0 * math.pi * np.arange(n_t) / max(n_t, 1) + rng.uniform(0, 2 * math.pi))
    rho = np.exp(-0.5 * ((z[None, :] - (mean_m + drift[:, None])) / sigma) ** 2)
    rho[:, rng.integers(0, n_z)] *= 1.0 + 0.5 * rng.uniform(0.0, 1.0, n_t)
    rho /= rho.sum(axis=1, keepdims=True)
    srcs = cfg.sources_of_wfs(wfs_index)
    xy = np.zeros((len(srcs), 2))
    if launch == "side":
        for i, s in enumerate(srcs):
            az = math.atan2(cfg.sources[s].theta_y_rad, cfg.sources[s].theta_x_rad)
            xy[i] = (cfg.pupil.r_out_m * math.cos(az), cfg.pupil.r_out_m * math.sin(az))
    return Sodium(wfs_index, z, rho, xy)


def linear_screen(n: int, c0: float, c_row: float, c_col: float) -> np.ndarray:
    """s[i][j] = c0 + c_row*i + c_col*j as float32 (pin input: bilinear of a linear screen)."""
    i = np.arange(n, dtype=np.float64)
    return (c0 + c_row * i[:, None] + c_col * i[None, :]).astype(np.float32)
