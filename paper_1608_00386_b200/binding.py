"""Thin ctypes binding of libao.so: same names as include/ao.h, argument marshalling only.

Every step of the forward model runs in the CUDA kernels behind the C ABI; this module
only converts torch tensors to device pointers and descriptors to C structs.  PyTorch is
used for device memory and streams.  There is no CPU fallback: if libao.so is missing or
there is no CUDA device, the calls raise.
"""
from __future__ import annotations

import ctypes as C
import math
import os
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libao.so")

AO_OK = 0
STATUS_NAMES = {0: "AO_OK", 1: "AO_ERR_INVALID_ARG", 2: "AO_ERR_SHAPE", 3: "AO_ERR_UNSUPPORTED",
                4: "AO_ERR_CUDA", 5: "AO_ERR_WORKSPACE"}

# every symbol include/ao.h declares
EXPORTS = ["ao_geometry_create", "ao_geometry_destroy", "ao_workspace_bytes", "ao_set_workspace",
           "ao_phase_elems_per_step", "ao_phase_offset", "ao_wfs_valid", "ao_trace_layers",
           "ao_sh_images", "ao_centroids", "ao_psf", "ao_psf_static", "ao_set_psf_band", "ao_psf_poly", "ao_set_phase_map", "ao_set_sodium", "ao_modes_to_map", "ao_strehl", "ao_strehl_marechal", "ao_forward", "ao_forward_host", "ao_probe_fp32", "ao_last_h2d_bytes", "ao_launch_count",
           "ao_last_error", "ao_version"]


class AoError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"{STATUS_NAMES.get(status, status)}: {message}")
        self.status = status


class ao_pupil(C.Structure):
    _fields_ = [("n", C.c_int32), ("pitch_m", C.c_double), ("amp_host", C.POINTER(C.c_float))]


class ao_wfs(C.Structure):
    _fields_ = [("n_sub", C.c_int32), ("n_samp", C.c_int32), ("fft", C.c_int32), ("bin", C.c_int32),
                ("n_pix", C.c_int32), ("min_illum", C.c_float), ("amp_host", C.POINTER(C.c_float))]


class ao_layer(C.Structure):
    _fields_ = [("n", C.c_int32), ("pitch_m", C.c_double), ("height_m", C.c_double),
                ("wind_x_mps", C.c_double), ("wind_y_mps", C.c_double), ("screen_dev", C.c_void_p)]


class ao_source(C.Structure):
    _fields_ = [("theta_x_rad", C.c_double), ("theta_y_rad", C.c_double), ("altitude_m", C.c_double),
                ("lambda_m", C.c_double), ("wfs_index", C.c_int32)]


class ao_noise(C.Structure):
    _fields_ = [("seed", C.c_uint64), ("photons_per_subap", C.c_float), ("read_noise_e", C.c_float)]


_lib = None


def load_library():
    """dlopen libao.so and declare the prototypes.  Fails loudly if the extension is not built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_1608_00386_b200.build` "
                          "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    vp, i32, i64, dbl, szt = C.c_void_p, C.c_int, C.c_int64, C.c_double, C.c_size_t
    L.ao_geometry_create.argtypes = [C.POINTER(ao_pupil), C.POINTER(ao_wfs), i32, C.POINTER(ao_layer), i32,
                                     C.POINTER(ao_source), i32, dbl, i32, C.POINTER(vp)]
    L.ao_geometry_destroy.argtypes = [vp]
    L.ao_workspace_bytes.argtypes = [vp, i32]; L.ao_workspace_bytes.restype = szt
    L.ao_set_workspace.argtypes = [vp, vp, szt]
    L.ao_phase_elems_per_step.argtypes = [vp]; L.ao_phase_elems_per_step.restype = szt
    L.ao_phase_offset.argtypes = [vp, i32, i32]; L.ao_phase_offset.restype = szt
    L.ao_wfs_valid.argtypes = [vp, i32, C.POINTER(C.c_uint8)]
    L.ao_trace_layers.argtypes = [vp, i64, i32, dbl, vp, vp]
    L.ao_sh_images.argtypes = [vp, i32, vp, i64, i32, dbl, C.POINTER(ao_noise), vp, vp, vp]
    L.ao_centroids.argtypes = [vp, i32, vp, i32, vp, vp]
    L.ao_psf.argtypes = [vp, vp, i64, i32, dbl, vp, i32, vp]
    L.ao_psf_static.argtypes = [vp, i32, vp, i32, vp, i32, vp]
    L.ao_set_psf_band.argtypes = [vp, C.POINTER(dbl), C.POINTER(dbl), i32]
    L.ao_psf_poly.argtypes = [vp, vp, i64, i32, dbl, vp, i32, vp]
    L.ao_set_phase_map.argtypes = [vp, i32, vp]
    L.ao_set_sodium.argtypes = [vp, i32, i32, C.POINTER(dbl), C.POINTER(dbl), i32, C.POINTER(dbl)]
    L.ao_modes_to_map.argtypes = [vp, vp, i32, i64, vp, C.c_float, vp, vp]
    L.ao_strehl.argtypes = [vp, vp, dbl, vp, vp]
    L.ao_strehl_marechal.argtypes = [vp, vp, i32, vp, vp]
    L.ao_forward.argtypes = [vp, i64, i32, dbl, C.POINTER(ao_noise), C.POINTER(vp), vp, i32, vp]
    L.ao_forward_host.argtypes = [vp, C.POINTER(vp), i64, i32, dbl, C.POINTER(ao_noise), C.POINTER(vp), vp, vp]
    L.ao_probe_fp32.argtypes = [vp, i32, C.POINTER(dbl)]
    L.ao_last_h2d_bytes.argtypes = [vp]; L.ao_last_h2d_bytes.restype = C.c_uint64
    L.ao_launch_count.argtypes = [vp]; L.ao_launch_count.restype = i64
    L.ao_last_error.restype = C.c_char_p
    L.ao_version.restype = C.c_char_p
    _lib = L
    return L


def _check(rc: int):
    if rc != AO_OK:
        raise AoError(rc, load_library().ao_last_error().decode())


def _ptr(t) -> Optional[int]:
    return None if t is None else int(t.data_ptr())


def _stream() -> int:
    import torch
    return int(torch.cuda.current_stream().cuda_stream)


def _noise(nz):
    if nz is None:
        return None
    return C.byref(ao_noise(int(nz.seed) & (2 ** 64 - 1), float(nz.photons_per_subap), float(nz.read_noise_e)))


class Geometry:
    """Owner of an ao_geometry handle (ao_geometry_create / ao_geometry_destroy).

    `cfg` is a paper_1608_00386_b200.inputs.Config; its screens are uploaded once into torch
    CUDA tensors that the handle borrows (kept alive here).  Methods mirror the C entry points.
    """

    def __init__(self, cfg, device: str = "cuda:0", workspace_steps: int = 1, screens=None):
        import torch
        self.lib = load_library()
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1608_00386_b200 needs a CUDA device (no CPU fallback)")
        self.cfg = cfg
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        if screens is None:
            screens = [l.screen_dev if getattr(l, "screen_dev", None) is not None else
                       torch.from_numpy(np.ascontiguousarray(l.screen, dtype=np.float32)).to(self.device)
                       for l in cfg.layers]
        self.screens = screens
        fp = C.POINTER(C.c_float)
        self._keep = []

        def hostf(a):
            a = np.ascontiguousarray(a, dtype=np.float32)
            self._keep.append(a)
            return a.ctypes.data_as(fp)

        pup = ao_pupil(cfg.pupil.n, cfg.pupil.pitch_m, hostf(cfg.pupil.amp))
        wfs = (ao_wfs * max(1, len(cfg.wfs)))(*[
            ao_wfs(w.n_sub, w.n_samp, w.fft, w.bin, w.n_pix, w.min_illum, hostf(w.amp)) for w in cfg.wfs])
        lay = (ao_layer * max(1, len(cfg.layers)))(*[
            ao_layer(l.n, l.pitch_m, l.height_m, l.wind_x_mps, l.wind_y_mps, int(s.data_ptr()))
            for l, s in zip(cfg.layers, screens)])
        src = (ao_source * max(1, len(cfg.sources)))(*[
            ao_source(s.theta_x_rad, s.theta_y_rad, s.altitude_m, s.lambda_m, s.wfs_index) for s in cfg.sources])
        h = C.c_void_p()
        _check(self.lib.ao_geometry_create(C.byref(pup), wfs, len(cfg.wfs), lay, len(cfg.layers), src,
                                           len(cfg.sources), cfg.lambda_ref_m, cfg.psf_fft, C.byref(h)))
        self.handle = h
        self.workspace = None
        self.phase_maps = {}
        self.set_workspace_steps(workspace_steps)
        for si, m in getattr(cfg, "phase_maps", {}).items():
            self.set_phase_map(si, m)
        if getattr(cfg, "sodium", None) is not None:
            self.set_sodium(cfg.sodium)
        if getattr(cfg, "psf_band", None) is not None:
            self.set_psf_band(*cfg.psf_band)

    # ---- lifetime ----
    def close(self):
        if getattr(self, "handle", None):
            self.lib.ao_geometry_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_phase_map(self, source: int, phase_map):
        """ao_set_phase_map: additive [N_s][N_s] phase map (numpy array, CUDA tensor, or None to clear)."""
        import torch
        if phase_map is None:
            self.phase_maps.pop(source, None)
            _check(self.lib.ao_set_phase_map(self.handle, int(source), None))
            return
        t = torch.as_tensor(np.ascontiguousarray(phase_map, dtype=np.float32) if isinstance(phase_map, np.ndarray)
                            else phase_map, dtype=torch.float32).to(self.device).contiguous()
        self.phase_maps[source] = t                      # borrowed by the library: keep it alive
        _check(self.lib.ao_set_phase_map(self.handle, int(source), _ptr(t)))

    def set_sodium(self, sodium):
        """ao_set_sodium: extended beacon of one WFS from an inputs.Sodium (None or n_z = 0 clears wfs 0's)."""
        dp = C.POINTER(C.c_double)
        if sodium is None:
            _check(self.lib.ao_set_sodium(self.handle, 0, 0, None, None, 0, None))
            return
        z = np.ascontiguousarray(sodium.z_m, dtype=np.float64)
        rho = np.ascontiguousarray(np.atleast_2d(sodium.rho), dtype=np.float64)
        xy = np.ascontiguousarray(sodium.launch_xy_m, dtype=np.float64)
        _check(self.lib.ao_set_sodium(self.handle, int(sodium.wfs_index), int(z.size), z.ctypes.data_as(dp),
                                      rho.ctypes.data_as(dp), int(rho.shape[0]), xy.ctypes.data_as(dp)))

    def modes_to_map(self, modes, coeffs, sign: float, out):
        """ao_modes_to_map: out[i] = sign * sum_m coeffs[m] modes[m][i] (CUDA float32 tensors; out is overwritten)."""
        n_modes = int(modes.shape[0]) if modes is not None else 0
        if modes is not None:
            modes, coeffs = modes.contiguous(), coeffs.contiguous()      # [n_modes][n_elems] row-major, as the ABI says
        assert out.is_contiguous()
        _check(self.lib.ao_modes_to_map(self.handle, _ptr(modes), n_modes, int(out.numel()), _ptr(coeffs),
                                        float(sign), _ptr(out), _stream()))
        return out

    # ---- sizes ----
    def workspace_bytes(self, max_steps: int) -> int:
        return int(self.lib.ao_workspace_bytes(self.handle, int(max_steps)))

    def set_workspace_steps(self, max_steps: int):
        import torch
        nbytes = self.workspace_bytes(max_steps)
        self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        _check(self.lib.ao_set_workspace(self.handle, _ptr(self.workspace), nbytes))

    def phase_elems_per_step(self) -> int:
        return int(self.lib.ao_phase_elems_per_step(self.handle))

    def phase_offset(self, source: int, step: int = 0) -> int:
        return int(self.lib.ao_phase_offset(self.handle, source, step))

    def wfs_valid(self, w: int) -> np.ndarray:
        W = self.cfg.wfs[w]
        v = np.zeros(W.n_sub * W.n_sub, dtype=np.uint8)
        n = self.lib.ao_wfs_valid(self.handle, w, v.ctypes.data_as(C.POINTER(C.c_uint8)))
        if n < 0:
            raise AoError(1, "ao_wfs_valid: bad index")
        return v

    def probe_fp32(self, packed: bool = False) -> float:
        """ao_probe_fp32: measured FP32 rate of an FMA-chain micro-kernel, TFLOP/s."""
        out = C.c_double(0.0)
        _check(self.lib.ao_probe_fp32(self.handle, int(bool(packed)), C.byref(out)))
        return float(out.value)

    def last_h2d_bytes(self) -> int:
        """ao_last_h2d_bytes: bytes of screens the last forward_host call uploaded."""
        return int(self.lib.ao_last_h2d_bytes(self.handle))

    def launch_count(self) -> int:
        return int(self.lib.ao_launch_count(self.handle))

    # ---- compute (asynchronous on torch's current stream) ----
    def trace_layers(self, step0: int, n_steps: int, dt_s: float, phase=None):
        import torch
        if phase is None:
            phase = torch.empty(n_steps * self.phase_elems_per_step(), dtype=torch.float32, device=self.device)
        _check(self.lib.ao_trace_layers(self.handle, step0, n_steps, dt_s, _ptr(phase), _stream()))
        return phase

    def phase_view(self, phase, source: int, step: int = 0):
        N = self.cfg.grid_n(source)
        o = self.phase_offset(source, step)
        return phase[o:o + N * N].view(N, N)

    def sh_images(self, w: int, phase, step0: int, n_steps: int, dt_s: float, noise=None,
                  want_images=True, want_slopes=True, images=None, slopes=None):
        import torch
        if not 0 <= w < len(self.cfg.wfs):       # let the library report the bad index
            _check(self.lib.ao_sh_images(self.handle, w, None, step0, n_steps, dt_s, None, None, None, _stream()))
        W = self.cfg.wfs[w]
        n_sel = len(self.cfg.sources_of_wfs(w))
        nsa = W.n_sub * W.n_sub
        if want_images and images is None:
            images = torch.empty((n_steps, n_sel, nsa, W.n_pix, W.n_pix), dtype=torch.float32, device=self.device)
        if want_slopes and slopes is None:
            slopes = torch.empty((n_steps, n_sel, 2, nsa), dtype=torch.float32, device=self.device)
        _check(self.lib.ao_sh_images(self.handle, w, _ptr(phase), step0, n_steps, dt_s, _noise(noise),
                                     _ptr(images), _ptr(slopes), _stream()))
        return images, slopes

    def centroids(self, w: int, images, slopes=None):
        import torch
        W = self.cfg.wfs[w]
        nsa = W.n_sub * W.n_sub
        n_sets = images.numel() // (nsa * W.n_pix * W.n_pix)
        if slopes is None:
            slopes = torch.empty((n_sets, 2, nsa), dtype=torch.float32, device=self.device)
        _check(self.lib.ao_centroids(self.handle, w, _ptr(images), n_sets, _ptr(slopes), _stream()))
        return slopes

    def psf(self, phase, step0: int, n_steps: int, dt_s: float, psf=None, accumulate=False):
        import torch
        M = self.cfg.psf_fft
        n_sci = len(self.cfg.science_sources())
        if psf is None:
            psf = torch.zeros((n_sci, M, M), dtype=torch.float32, device=self.device)
        _check(self.lib.ao_psf(self.handle, _ptr(phase), step0, n_steps, dt_s, _ptr(psf), int(accumulate), _stream()))
        return psf

    def psf_static(self, direction: int, phase, n_steps: int, psf, accumulate=False):
        """ao_psf_static: PSF of one science direction with the FFT intermediate in the library's static device array
        (no workspace, no allocation).  `psf` [M][M] is caller-owned: this binding allocates nothing either."""
        _check(self.lib.ao_psf_static(self.handle, int(direction), _ptr(phase), int(n_steps), _ptr(psf), int(accumulate), _stream()))
        return psf

    def set_psf_band(self, lambdas_m=None, weights=None):
        """ao_set_psf_band: wavelengths [m] and weights of the polychromatic PSF (None clears the band)."""
        dp = C.POINTER(C.c_double)
        if lambdas_m is None:
            _check(self.lib.ao_set_psf_band(self.handle, None, None, 0))
            return
        lam = np.ascontiguousarray(lambdas_m, dtype=np.float64); w = np.ascontiguousarray(weights, dtype=np.float64)
        assert lam.shape == w.shape
        _check(self.lib.ao_set_psf_band(self.handle, lam.ctypes.data_as(dp), w.ctypes.data_as(dp), int(lam.size)))

    def psf_poly(self, phase, step0: int, n_steps: int, dt_s: float, psf=None, accumulate=False):
        """ao_psf_poly: polychromatic long-exposure PSF over the band set with set_psf_band."""
        import torch
        M = self.cfg.psf_fft
        if psf is None:
            psf = torch.zeros((len(self.cfg.science_sources()), M, M), dtype=torch.float32, device=self.device)
        _check(self.lib.ao_psf_poly(self.handle, _ptr(phase), step0, n_steps, dt_s, _ptr(psf), int(accumulate), _stream()))
        return psf

    def strehl(self, psf, n_exposures: float):
        """ao_strehl: [n_sci] Strehl ratios of a long-exposure PSF summed over n_exposures steps."""
        import torch
        out = torch.empty((len(self.cfg.science_sources()),), dtype=torch.float32, device=self.device)
        _check(self.lib.ao_strehl(self.handle, _ptr(psf), float(n_exposures), _ptr(out), _stream()))
        return out

    def strehl_marechal(self, phase, n_steps: int):
        """ao_strehl_marechal: [n_steps][n_sci] exp(-weighted phase variance) from an ao_trace_layers phase buffer."""
        import torch
        out = torch.empty((n_steps, len(self.cfg.science_sources())), dtype=torch.float32, device=self.device)
        _check(self.lib.ao_strehl_marechal(self.handle, _ptr(phase), int(n_steps), _ptr(out), _stream()))
        return out

    def forward(self, step0: int, n_steps: int, dt_s: float, slopes: Sequence, psf=None, accumulate=False, noise=None):
        """ao_forward: every WFS (slopes[w] device tensors, None to skip) and the science PSF in one call."""
        nw = len(self.cfg.wfs)
        sl = (C.c_void_p * max(1, nw))(*[(_ptr(t) if t is not None else None) for t in slopes])
        _check(self.lib.ao_forward(self.handle, step0, n_steps, dt_s, _noise(noise), sl, _ptr(psf),
                                   int(accumulate), _stream()))

    def forward_host(self, step0: int, n_steps: int, dt_s: float, slopes_host: Sequence, psf_host=None,
                     screens_host: Optional[Sequence] = None, noise=None):
        """ao_forward_host: host (pinned) torch tensors in/out; copies are inside the call."""
        nw = len(self.cfg.wfs)
        sl = (C.c_void_p * max(1, nw))(*[(_ptr(t) if t is not None else None) for t in slopes_host])
        sc = None
        if screens_host is not None:
            sc = (C.c_void_p * len(screens_host))(*[_ptr(t) for t in screens_host])
        _check(self.lib.ao_forward_host(self.handle, sc, step0, n_steps, dt_s, _noise(noise), sl,
                                        _ptr(psf_host), _stream()))
