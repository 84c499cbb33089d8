"""GPU-vs-oracle parity at the sizes BASELINE.json states (pytest -m gpu).

Every workload runs at its full size on the GPU, through the same C-ABI entry points and in the launch
configuration bench.py times (ao_forward, 50 steps per call for c4).  The FP64 oracle then recomputes a bounded
subset (some sources, some steps) so that it stays in seconds per case: the GPU arrays are compared element by
element on that subset.  Beside the array-level relative L2 (the bar of north_star) the per-subaperture maximum
relative L2 is measured and written to gpurun_out/parity_report.jsonl (SURVEY.md section 8(c) "Parity bars").

Sizes: c1 80x80 subapertures of 12 samples, FFT 24, 3 screens of 2048^2; c2 6 LGS x 80x80 x FFT 32, 10 screens of
2048^2, with and without detector noise; c3 adds 3 NGS sensors (FFT 1024) and 10 science PSFs (FFT 2048);
c4 35 screens of 8192^2 (generated on the GPU as bench.py does), LGS FFT 16 / 32 / 64, steps 0, 499, 999.
"""
import math

import numpy as np
import pytest

import oracle
from paper_1608_00386_b200 import inputs
from tests.parity_util import (IMAGE_TOL, PHASE_TOL, SLOPE_TOL, check_wfs, per_subap_max_rel_l2, rel_l2, report)

pytestmark = pytest.mark.gpu


def _geo(cfg, steps=1):
    from paper_1608_00386_b200 import binding
    return binding.Geometry(cfg, workspace_steps=steps)


# ------------------------------------------------------------------------------------------------ c1
def test_c1_full_size_two_steps():
    """c1 as stated: 960^2 annular pupil, 80x80 subapertures, n = 12, FFT 24 (the 3 x 8 kernel), 6x6 pixels, three
    2048^2 screens, wind 0.5 px per step.  Both the phase-buffer path and the fused path, all subapertures."""
    import torch
    cfg = inputs.make_config(1, n_steps=2)
    assert cfg.wfs[0].n_sub == 80 and cfg.wfs[0].fft == 24 and cfg.layers[0].n == 2048 and cfg.pupil.n == 960
    ref = oracle.forward(cfg, 37, 2)
    geo = _geo(cfg, 2)
    phase = geo.trace_layers(37, 2, cfg.dt_s)
    img, slp = geo.sh_images(0, phase, 37, 2, cfg.dt_s)
    img_f, slp_f = geo.sh_images(0, None, 37, 2, cfg.dt_s)
    torch.cuda.synchronize()
    e_ph = max(rel_l2(geo.phase_view(phase, 0, k).cpu().numpy(), ref["phase"][0][k]) for k in range(2))
    assert e_ph <= PHASE_TOL, e_ph
    assert np.array_equal(geo.wfs_valid(0), ref["valid"][0])
    a = check_wfs(cfg, geo, ref, 0, img, slp, 2, "c1 full, phase buffer")
    b = check_wfs(cfg, geo, ref, 0, img_f, slp_f, 2, "c1 full, phase_dev = NULL")
    report("c1_full", phase_rel_l2=e_ph, images_rel_l2=max(a[0], b[0]), slopes_max_abs=max(a[1], b[1]),
           per_subap_rel_l2=max(a[2], b[2]), valid_subaps=int(ref["valid"][0].sum()))


# ------------------------------------------------------------------------------------------------ c2
@pytest.fixture(scope="module")
def c2_full():
    cfg = inputs.make_config(2, n_steps=1)
    assert cfg.wfs[0].n_sub == 80 and cfg.layers[0].n == 2048 and len(cfg.layers) == 10 and len(cfg.sources) == 6
    return cfg


def test_c2_full_size_noiseless_all_six_lgs(c2_full):
    """c2 as stated, one step, all six LGS in full: fused kernel k_fused<32> (cone effect, 10 layers) against the
    oracle, and the traced phase of every LGS through ao_trace_layers."""
    import torch
    cfg = c2_full
    step = 50
    ref = oracle.forward(cfg, step, 1)
    geo = _geo(cfg, 1)
    phase = geo.trace_layers(step, 1, cfg.dt_s)
    img, slp = geo.sh_images(0, None, step, 1, cfg.dt_s)
    img_p, slp_p = geo.sh_images(0, phase, step, 1, cfg.dt_s)
    torch.cuda.synchronize()
    e_ph = max(rel_l2(geo.phase_view(phase, s, 0).cpu().numpy(), ref["phase"][s][0]) for s in range(6))
    assert e_ph <= PHASE_TOL, e_ph
    a = check_wfs(cfg, geo, ref, 0, img, slp, 1, "c2 full fused")
    b = check_wfs(cfg, geo, ref, 0, img_p, slp_p, 1, "c2 full from the phase buffer")
    report("c2_full_noiseless", phase_rel_l2=e_ph, images_rel_l2=max(a[0], b[0]), slopes_max_abs=max(a[1], b[1]),
           per_subap_rel_l2=max(a[2], b[2]))


def _noise_protocol(cfg, ref, noisy, slopes, step_index, w=0):
    """Reading O5: identical Poisson counts on >= 1 - 1e-5 of the pixels, slopes within
    1e-4 px on the subapertures whose counts all agree, residual mean / variance within 4 sigma."""
    ron = cfg.noise.read_noise_e
    tot = bad = 0
    worst = 0.0
    resid, var = [], []
    v = ref["valid"][w].astype(bool)
    for si, s in enumerate(cfg.sources_of_wfs(w)):
        g = noisy[step_index, si].cpu().numpy().astype(np.float64)
        r = ref["noisy"][s][0]
        same = np.abs(g - r) < 0.5                          # the Gaussian part is continuous: same Poisson count
        tot += int(same[v].size); bad += int((~same[v]).sum())
        ok_sub = same.reshape(same.shape[0], -1).all(axis=1) & v
        assert np.all(np.abs(g - r)[same] <= 2e-3 + 1e-6 * np.abs(r)[same])     # fp32 Box-Muller and fp32 storage against fp64
        assert np.all(g[~v] == 0.0)
        d = np.abs(slopes[step_index, si].cpu().numpy().astype(np.float64) - ref["slopes"][s][0])
        worst = max(worst, d[:, ok_sub].max())
        mu = cfg.noise.photons_per_subap * ref["images"][s][0]
        resid.append((g - mu)[v].ravel()); var.append((mu + ron ** 2)[v].ravel())
    assert bad <= max(1, int(1e-5 * tot)), f"{bad} of {tot} Poisson counts differ"
    assert worst <= SLOPE_TOL, worst
    resid = np.concatenate(resid); var = np.concatenate(var)
    assert abs(resid.sum() / math.sqrt(var.sum())) < 4.0
    assert abs((resid ** 2 / var).mean() - 1.0) < 4.0 * math.sqrt(2.5 / resid.size)
    return bad, tot, worst


def test_c2_full_size_noise_through_the_fused_kernel_and_ao_forward(c2_full):
    """c2's real hot path: detector noise inside the fused kernel (phase_dev = NULL, noise = cfg.noise:
    k_fused<32, NOISE>), all six LGS at 80x80, and the same through ao_forward(noise = ...)."""
    import torch
    cfg = c2_full
    step = 99
    ref = oracle.forward(cfg, step, 1, want_phase=False, noise_on=True)
    geo = _geo(cfg, 2)
    noisy, slopes = geo.sh_images(0, None, step, 1, cfg.dt_s, noise=cfg.noise)
    torch.cuda.synchronize()
    bad, tot, worst = _noise_protocol(cfg, ref, noisy, slopes, 0)
    # ao_forward with noise: steps 98 and 99 in one call (slopes only).  Step 99 is now the second step of its CTA
    # pair (it was the first above): same counts up to the protocol, not bit-identical.  Step 98 against the oracle too.
    sl = [torch.full((2, 6, 2, 6400), float("nan"), dtype=torch.float32, device="cuda")]
    geo.forward(step - 1, 2, cfg.dt_s, sl, psf=None, noise=cfg.noise)
    torch.cuda.synchronize()
    # a flipped Poisson count moves the two slopes of one subaperture; the protocol allows 1e-5 of the pixels to flip
    d99 = (sl[0][1] - slopes[0]).abs()
    allowed = 2 * max(1, int(1e-5 * tot))
    assert int((d99 > 1e-5).sum()) <= allowed, "ao_forward(noise) and ao_sh_images(noise) disagree on more than Poisson flips"
    ref98 = oracle.forward(cfg, step - 1, 1, want_phase=False, noise_on=True)
    worst98 = 0.0
    n_off = 0
    for si, s in enumerate(cfg.sources_of_wfs(0)):
        d = np.abs(sl[0][0, si].cpu().numpy().astype(np.float64) - ref98["slopes"][s][0])
        n_off += int((d > SLOPE_TOL).sum())
        worst98 = max(worst98, float(np.median(d)))
    assert n_off <= allowed and worst98 <= 1e-5, (n_off, worst98)  # a flipped count moves one subaperture's slopes
    report("c2_full_noise", counts_differing=bad, counts_total=tot, slopes_max_abs_on_equal_counts=worst,
           forward_slopes_off=n_off)


def test_c2_full_size_lgs_elongation(c2_full):
    """NEXT-3 at c2's full size: an extended sodium layer (5 scatterers, side launch, time-varying profile) through the
    fused kernel, LGS 0 and LGS 3 in full against the oracle."""
    import torch
    cfg = c2_full
    cfg.sodium = inputs.sodium_profile(cfg, n_z=5, n_t=8, launch="side")
    try:
        ref = oracle.forward(cfg, 13, 1, want_phase=False, sources=[0, 3])
        geo = _geo(cfg, 1)
        img, slp = geo.sh_images(0, None, 13, 1, cfg.dt_s)
        torch.cuda.synchronize()
        a = check_wfs(cfg, geo, ref, 0, img, slp, 1, "c2 full, elongated spots", sources=[0, 3])
        report("c2_full_elongation", images_rel_l2=a[0], slopes_max_abs=a[1], per_subap_rel_l2=a[2])
    finally:
        cfg.sodium = None


# ------------------------------------------------------------------------------------------------ c3
def test_c3_full_size_ngs_sensors_and_two_science_psfs():
    """c3 as stated, one step: the three NGS sensors (2x2 subapertures of 480 samples, FFT 1024, 128x128 pixels) in
    full, and two of the ten science PSFs (960^2 pupil, FFT 2048): the (-30", -30") corner and the (45", 45")
    direction; the LGS sensors of c3 are those of c2 (checked above) and are compared on LGS 1 and 4 here, all through
    ao_forward-equivalent separate calls plus one ao_forward call for the slopes and the PSFs."""
    import torch
    cfg = inputs.make_config(3, n_steps=1)
    assert cfg.wfs[1].fft == 1024 and cfg.wfs[1].n_samp == 480 and cfg.psf_fft == 2048
    sci = cfg.science_sources()
    assert len(sci) == 10
    subset = [1, 4] + cfg.sources_of_wfs(1) + [sci[0], sci[9]]
    step = 25
    ref = oracle.forward(cfg, step, 1, want_phase=False, sources=subset)
    geo = _geo(cfg, 1)
    img_n, slp_n = geo.sh_images(1, None, step, 1, cfg.dt_s)
    img_l, slp_l = geo.sh_images(0, None, step, 1, cfg.dt_s)
    psf = geo.psf(None, step, 1, cfg.dt_s)
    torch.cuda.synchronize()
    a = check_wfs(cfg, geo, ref, 1, img_n, slp_n, 1, "c3 full NGS")
    b = check_wfs(cfg, geo, ref, 0, img_l, slp_l, 1, "c3 full LGS", sources=[1, 4])
    e_psf = max(rel_l2(psf[di].cpu().numpy(), ref["psf"][sci[di]]) for di in (0, 9))
    assert e_psf <= IMAGE_TOL, e_psf
    for di in range(10):
        assert abs(float(psf[di].sum(dtype=torch.float64)) - 1.0) < 1e-4          # Parseval for all ten
    # the whole step in one call
    sl = [torch.empty_like(slp_l), torch.empty_like(slp_n)]
    p2 = torch.zeros_like(psf)
    geo.forward(step, 1, cfg.dt_s, sl, psf=p2)
    torch.cuda.synchronize()
    assert torch.equal(sl[0], slp_l) and torch.equal(sl[1], slp_n)
    assert torch.allclose(p2, psf, rtol=1e-6, atol=0.0)
    strehl = geo.strehl(psf, 1).cpu().numpy()
    want = np.array([oracle.strehl(ref["psf"][sci[di]], cfg.pupil.amp, 1) for di in (0, 9)])
    assert np.abs(strehl[[0, 9]] - want).max() <= 1e-5 * max(1.0, np.abs(want).max())
    report("c3_full", ngs_images_rel_l2=a[0], ngs_slopes_max_abs=a[1], ngs_per_subap_rel_l2=a[2],
           lgs_images_rel_l2=b[0], lgs_slopes_max_abs=b[1], lgs_per_subap_rel_l2=b[2], psf_rel_l2=e_psf)


# ------------------------------------------------------------------------------------------------ c4
@pytest.fixture(scope="module")
def c4_screens():
    """The 35 screens of 8192^2 of c4, generated on the GPU exactly as bench.py does, with host copies for the oracle."""
    import torch
    cfg = inputs.make_config(4, lgs_fft=32, device="cuda:0", keep_on_device=True)
    assert len(cfg.layers) == 35 and cfg.layers[0].n == 8192
    inputs.screens_to_host(cfg)
    torch.cuda.synchronize()
    return cfg.layers


def _c4(layers, M):
    cfg = inputs.make_config(4, lgs_fft=M, with_screens=False)
    for lay, full in zip(cfg.layers, layers):
        assert (lay.height_m, lay.wind_x_mps, lay.wind_y_mps, lay.weight) == \
               (full.height_m, full.wind_x_mps, full.wind_y_mps, full.weight)
        lay.screen, lay.screen_dev = full.screen, full.screen_dev
    return cfg


@pytest.mark.parametrize("M", [32, 16, 64])
def test_c4_full_size_lgs_steps_0_499_999(c4_screens, M):
    """c4 at full size (80x80 subapertures, 8192^2 screens, 35 layers) for every LGS FFT size of the sweep, in the
    configuration bench.py times: ao_forward over 50-step batches.  Steps 0, 499 and 999 are
    compared with the oracle on LGS 0 and LGS 3 in full: slopes from ao_forward, images and slopes from ao_sh_images.
    This is where the 32.32 fixed-point column coordinates and FP64 origins see 8192-pixel screens, where M = 16 work
    items hold more than 16 subapertures (second column half of the fused tile), and where step pairs start odd."""
    import torch
    cfg = _c4(c4_screens, M)
    lgs, ngs = cfg.wfs
    assert lgs.n_sub == 80 and lgs.fft == M and lgs.n_samp == M // 2
    geo = _geo(cfg, 50)
    sl = [torch.empty((50, 6, 2, 6400), dtype=torch.float32, device="cuda"),
          torch.empty((50, 3, 2, 4), dtype=torch.float32, device="cuda")]
    psf = torch.zeros((1, cfg.psf_fft, cfg.psf_fft), dtype=torch.float32, device="cuda")
    pick = [0, 3]
    worst = [0.0, 0.0, 0.0]
    for f0, idx in ((0, 0), (450, 49), (950, 49)):
        step = f0 + idx
        ref = oracle.forward(cfg, step, 1, want_phase=False, want_psf=False, sources=pick)
        for t in sl:
            t.fill_(float("nan"))
        geo.forward(f0, 50, cfg.dt_s, sl, psf=psf, accumulate=False)
        img, slp = geo.sh_images(0, None, step, 2, cfg.dt_s)        # a pair that starts on an odd step for 499 / 999
        torch.cuda.synchronize()
        assert not torch.isnan(sl[0]).any() and not torch.isnan(sl[1]).any()
        r = check_wfs(cfg, geo, ref, 0, img, slp, 1, f"c4 M={M} step {step} ao_sh_images", sources=pick)
        r2 = check_wfs(cfg, geo, ref, 0, None, sl[0], 1, f"c4 M={M} step {step} ao_forward", sources=pick, steps=[idx])
        assert float((sl[0][idx] - slp[0]).abs().max()) <= 2e-5      # same step as first / second of its CTA pair
        worst = [max(worst[0], r[0]), max(worst[1], r[1], r2[1]), max(worst[2], r[2])]
    assert np.array_equal(geo.wfs_valid(0), ref["valid"][0])
    report(f"c4_full_M{M}", images_rel_l2=worst[0], slopes_max_abs=worst[1], per_subap_rel_l2=worst[2],
           valid_subaps=int(ref["valid"][0].sum()))


def test_c4_full_size_ngs_sensor_and_science_psf(c4_screens):
    """The rest of the c4 step at full size: the three NGS sensors (FFT 1024) at step 999 and the on-axis science PSF
    (FFT 2048) summed over steps 499 and 500, both from 8192^2 screens, against the oracle."""
    import torch
    cfg = _c4(c4_screens, 32)
    ngs_src, sci = cfg.sources_of_wfs(1), cfg.science_sources()
    geo = _geo(cfg, 2)
    ref = oracle.forward(cfg, 999, 1, want_phase=False, want_psf=False, sources=ngs_src)
    img, slp = geo.sh_images(1, None, 999, 1, cfg.dt_s)
    torch.cuda.synchronize()
    a = check_wfs(cfg, geo, ref, 1, img, slp, 1, "c4 NGS step 999")
    refp = oracle.forward(cfg, 499, 2, want_phase=False, want_wfs=False, sources=sci)
    psf = geo.psf(None, 499, 2, cfg.dt_s)
    torch.cuda.synchronize()
    e = rel_l2(psf[0].cpu().numpy(), refp["psf"][sci[0]])
    assert e <= IMAGE_TOL, e
    report("c4_full_ngs_psf", ngs_images_rel_l2=a[0], ngs_slopes_max_abs=a[1], ngs_per_subap_rel_l2=a[2], psf_rel_l2=e)


def test_c4_full_size_polychromatic_psf(c4_screens):
    """NEXT-4 at full size: the on-axis science PSF of c4 (960^2 pupil, 2048^2 pixels, chirp-z FFTs of 4096) over a
    two-wavelength band, one step from the 8192^2 screens, against the oracle."""
    import torch
    cfg = _c4(c4_screens, 32)
    cfg.psf_band = ([2.0e-6, 2.4e-6], [0.5, 0.5])
    sci = cfg.science_sources()
    refp = oracle.forward(cfg, 123, 1, want_phase=False, want_wfs=False, sources=sci)
    geo = _geo(cfg, 1)
    psf = geo.psf_poly(None, 123, 1, cfg.dt_s)
    torch.cuda.synchronize()
    e = rel_l2(psf[0].cpu().numpy(), refp["psf"][sci[0]])
    assert e <= IMAGE_TOL, e
    report("c4_full_psf_poly", psf_rel_l2=e)


# ------------------------------------------------------------------------------------------------ fallbacks
def test_big_fft_generic_fallback_and_noise_on_a_big_sensor():
    """(i) A big-FFT sensor whose bin factor is not a power of two (beta = 6, FFT 128, 20x20 pixels of the central
    120) is outside the Stockham fast path and runs k_fft_big_generic.cu; (ii) detector noise on a big-FFT sensor runs
    the stand-alone k_noise on bright pixels (mu up to thousands: the mode-centred Poisson search)."""
    import torch
    cfg = inputs.make_config(3, n_sub=8, screen_n=512, n_steps=2)
    ngs = cfg.wfs[1]
    assert ngs.fft == 128
    ngs.bin, ngs.n_pix = 6, 20
    srcs = cfg.sources_of_wfs(1)
    ref = oracle.forward(cfg, 2, 2, want_phase=False, want_psf=False, sources=srcs)
    geo = _geo(cfg, 2)
    img, slp = geo.sh_images(1, None, 2, 2, cfg.dt_s)
    phase = geo.trace_layers(2, 2, cfg.dt_s)
    img_p, slp_p = geo.sh_images(1, phase, 2, 2, cfg.dt_s)
    torch.cuda.synchronize()
    a = check_wfs(cfg, geo, ref, 1, img, slp, 2, "generic big FFT, beta 6")
    check_wfs(cfg, geo, ref, 1, img_p, slp_p, 2, "generic big FFT from a phase buffer")
    # (ii) power-of-two bins again (fast path) with noise: 2e5 photons per subaperture
    cfg2 = inputs.make_config(3, n_sub=8, screen_n=512, n_steps=1)
    cfg2.noise = inputs.Noise(seed=77, photons_per_subap=2.0e5, read_noise_e=3.0)
    ref2 = oracle.forward(cfg2, 5, 1, want_phase=False, want_psf=False, noise_on=True, sources=srcs)
    geo2 = _geo(cfg2, 1)
    noisy, slopes = geo2.sh_images(1, None, 5, 1, cfg2.dt_s, noise=cfg2.noise)
    torch.cuda.synchronize()
    assert max(ref2["counts"][s].max() for s in srcs) > 1000          # bright pixels are exercised
    bad, tot, worst = _noise_protocol(cfg2, ref2, noisy, slopes, 0, w=1)
    report("generic_big_fft_and_big_noise", images_rel_l2=a[0], per_subap_rel_l2=a[2], counts_differing=bad,
           counts_total=tot)
