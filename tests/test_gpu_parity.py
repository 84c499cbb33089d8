"""GPU-vs-oracle parity through the C ABI (pytest -m gpu; runs on the B200 box).

Sizes are chosen so the FP64 oracle finishes in seconds while the inputs still span several
CTAs/tiles and ragged tails (subaperture grids that are not multiples of the CTA batch,
pupils not multiples of 32).  Tolerances: BASELINE.json north_star (tests/parity_util.py).
"""
import math

import numpy as np
import pytest

import oracle
from paper_1608_00386_b200 import inputs
from tests.parity_util import IMAGE_TOL, PHASE_TOL, SLOPE_TOL, check_wfs, rel_l2

pytestmark = pytest.mark.gpu


def _geo(cfg, steps=1):
    from paper_1608_00386_b200 import binding
    return binding.Geometry(cfg, workspace_steps=steps)


def _run_all(cfg, n_steps, step0=0):
    """Unfused API path: trace -> phase -> sh_images / psf.  Returns torch outputs."""
    import torch
    geo = _geo(cfg, n_steps)
    phase = geo.trace_layers(step0, n_steps, cfg.dt_s)
    out = {"phase": phase, "geo": geo, "images": {}, "slopes": {}}
    for w in range(len(cfg.wfs)):
        if cfg.sources_of_wfs(w):
            out["images"][w], out["slopes"][w] = geo.sh_images(w, phase, step0, n_steps, cfg.dt_s)
    if cfg.psf_fft and cfg.science_sources():
        out["psf"] = geo.psf(phase, step0, n_steps, cfg.dt_s)
    torch.cuda.synchronize()
    return out


def _check_phase(cfg, geo, phase, ref, n_steps):
    worst = 0.0
    for s in range(len(cfg.sources)):
        for k in range(n_steps):
            got = geo.phase_view(phase, s, k).cpu().numpy()
            worst = max(worst, rel_l2(got, ref["phase"][s][k]))
    assert worst <= PHASE_TOL, f"phase rel L2 {worst:.3e}"
    return worst


def _check_all(cfg, n_steps, step0=0):
    ref = oracle.forward(cfg, step0, n_steps)
    out = _run_all(cfg, n_steps, step0)
    geo = out["geo"]
    _check_phase(cfg, geo, out["phase"], ref, n_steps)
    for w in out["images"]:
        assert np.array_equal(geo.wfs_valid(w), ref["valid"][w])
        check_wfs(cfg, geo, ref, w, out["images"][w], out["slopes"][w], n_steps, cfg.name)
    if "psf" in out:
        for di, s in enumerate(cfg.science_sources()):
            e = rel_l2(out["psf"][di].cpu().numpy(), ref["psf"][s])
            assert e <= IMAGE_TOL, f"psf rel L2 {e:.3e}"
    # fused path (phase_dev = NULL): same outputs without a phase buffer
    for w in out["images"]:
        img, slp = geo.sh_images(w, None, step0, n_steps, cfg.dt_s)
        check_wfs(cfg, geo, ref, w, img, slp, n_steps, cfg.name + " fused")
        _, slp2 = geo.sh_images(w, None, step0, n_steps, cfg.dt_s, want_images=False)
        check_wfs(cfg, geo, ref, w, None, slp2, n_steps, cfg.name + " fused slopes-only")
    if "psf" in out:
        p2 = geo.psf(None, step0, n_steps, cfg.dt_s)
        for di, s in enumerate(cfg.science_sources()):
            assert rel_l2(p2[di].cpu().numpy(), ref["psf"][s]) <= IMAGE_TOL
    return out, ref


def test_c0_tiny_ngs_scao_full():
    cfg = inputs.make_config(0)
    _check_all(cfg, 1)


def test_c1_elt_ngs_scao_reduced_three_steps():
    # M = 24 (not a power of two), annular pupil, 3 layers, sub-pixel wind shift of 0.5 px/step
    cfg = inputs.make_config(1, n_sub=18, screen_n=512, n_steps=3)
    _check_all(cfg, 3, step0=5)


def test_c2_maory_lgs_reduced_noiseless():
    # 6 LGS with cone effect, 10 layers, off-axis, n_sub = 14 (ragged against any CTA batch)
    cfg = inputs.make_config(2, n_sub=14, screen_n=512, n_steps=2)
    _check_all(cfg, 2, step0=49)


def test_c3_full_mcao_reduced_long_exposure():
    # LGS + NGS (big FFT path, M = 128) + 10 science PSFs (M = 256) accumulated over 3 steps
    cfg = inputs.make_config(3, n_sub=8, screen_n=512, n_steps=3)
    assert cfg.wfs[1].fft == 128 and cfg.psf_fft == 256
    _check_all(cfg, 3)


@pytest.mark.parametrize("M", [16, 32, 64])
def test_c4_throughput_sweep_reduced(M):
    cfg = inputs.make_config(4, n_sub=10, screen_n=1024, n_steps=2, lgs_fft=M)
    assert len(cfg.layers) == 35
    _check_all(cfg, 2, step0=499)


def test_c2_noise_protocol():
    """Reading O5: identical Poisson counts on >= 1-1e-5 of the pixels; slopes within 1e-4 on
    subapertures whose counts all agree; residual statistics match Poisson + read noise."""
    import torch
    cfg = inputs.make_config(2, n_sub=14, screen_n=512, n_steps=2)
    n_steps = 2
    ref = oracle.forward(cfg, 0, n_steps, want_psf=False, noise_on=True)
    geo = _geo(cfg, n_steps)
    phase = geo.trace_layers(0, n_steps, cfg.dt_s)
    clean, _ = geo.sh_images(0, phase, 0, n_steps, cfg.dt_s)
    noisy, slopes = geo.sh_images(0, phase, 0, n_steps, cfg.dt_s, noise=cfg.noise)
    torch.cuda.synchronize()
    ron = cfg.noise.read_noise_e
    tot = bad = 0
    worst = 0.0
    resid, var = [], []
    for si, s in enumerate(cfg.sources_of_wfs(0)):
        for k in range(n_steps):
            g = noisy[k, si].cpu().numpy().astype(np.float64)
            r = ref["noisy"][s][k]
            # the Gaussian part is continuous: |g - r| < 0.5 <=> same Poisson count
            same = np.abs(g - r) < 0.5
            tot += same.size; bad += int((~same).sum())
            ok_sub = same.reshape(same.shape[0], -1).all(axis=1)
            assert np.abs(g - r)[same].max() < 2e-3            # fp32 Box-Muller vs fp64
            d = np.abs(slopes[k, si].cpu().numpy().astype(np.float64) - ref["slopes"][s][k])
            worst = max(worst, d[:, ok_sub].max())
            mu = cfg.noise.photons_per_subap * ref["images"][s][k]
            v = ref["valid"][0].astype(bool)
            resid.append((g - mu)[v].ravel()); var.append((mu + ron ** 2)[v].ravel())
    assert bad <= max(1, int(1e-5 * tot)), f"{bad} of {tot} Poisson counts differ"
    assert worst <= SLOPE_TOL
    resid = np.concatenate(resid); var = np.concatenate(var)
    assert abs(resid.sum() / math.sqrt(var.sum())) < 4.0
    assert abs((resid ** 2 / var).mean() - 1.0) < 4.0 * math.sqrt(2.5 / resid.size)
    # stand-alone noise path == fused path is not required; noiseless images unchanged
    check_wfs(cfg, geo, ref, 0, clean, None, n_steps, "c2 clean")


def test_noise_device_philox_matches_oracle_bits():
    """Bright flat images, no read noise: GPU Poisson counts must equal the oracle's exactly
    (same Philox words, same FP64 inverse-CDF search)."""
    import torch
    cfg = inputs.make_config(0, with_screens=False)
    cfg.layers[0].screen = np.zeros((256, 256), np.float32)
    nz = inputs.Noise(seed=0xDEADBEEF12345678, photons_per_subap=5000.0, read_noise_e=0.0)
    geo = _geo(cfg, 1)
    noisy, _ = geo.sh_images(0, None, 7, 1, cfg.dt_s, noise=nz)
    torch.cuda.synchronize()
    img, valid = oracle.sh_images(np.zeros((80, 80)), cfg.wfs[0].amp, 10, 8, 16, 2, 8, 0.5)
    _, counts = oracle.noise(img, valid, nz.seed, 0, 7, nz.photons_per_subap, 0.0)
    got = noisy[0, 0].cpu().numpy()
    assert np.array_equal(got[valid.astype(bool)], counts[valid.astype(bool)].astype(np.float32))
    assert counts.max() > 900      # mu ~ 1026 in the centre pixels: exp(-mu) underflows fp32


def test_centroids_standalone_matches_oracle():
    import torch
    cfg = inputs.make_config(0, with_screens=False)
    cfg.layers[0].screen = np.zeros((256, 256), np.float32)
    geo = _geo(cfg, 1)
    rng = np.random.default_rng(5)
    imgs = rng.uniform(0.0, 1.0, (3, 100, 8, 8)).astype(np.float32)
    imgs[1, 4] = 0.0                                    # zero-sum image -> slopes 0
    s = geo.centroids(0, torch.from_numpy(imgs).cuda())
    torch.cuda.synchronize()
    valid = geo.wfs_valid(0)
    for k in range(3):
        ref = oracle.centroids(imgs[k].astype(np.float64), valid)
        assert np.abs(s[k].cpu().numpy() - ref).max() <= 2e-6
    assert float(s[1, 0, 4]) == 0.0 and float(s[1, 1, 4]) == 0.0


def test_flat_wavefront_gives_zero_slopes_and_closed_form_image():
    import torch
    cfg = inputs.make_config(2, n_sub=6, screen_n=256, n_steps=1, with_screens=False)
    for l in cfg.layers:
        l.screen = np.full((256, 256), 3.25, np.float32)        # piston only
    geo = _geo(cfg, 1)
    img, slp = geo.sh_images(0, None, 0, 1, cfg.dt_s)
    torch.cuda.synchronize()
    valid = geo.wfs_valid(0).astype(bool)
    assert float(slp.abs().max()) <= 2e-6
    full = cfg.wfs[0].amp.reshape(6, 16, 6, 16).transpose(0, 2, 1, 3).reshape(36, 256).sum(1) == 256
    prof = np.array([0.004116392250, 0.005814901476, 0.013954378208, 0.476114328066])
    prof = np.concatenate([prof, prof[::-1]])                   # SURVEY.md section 8(c) c2 profile
    got = img[0, 0].cpu().numpy()[full]
    assert got.shape[0] > 0 and np.abs(got - np.outer(prof, prof)).max() < 2e-6
    assert np.all(img[0, :, ~valid].cpu().numpy() == 0.0)


def test_integer_pixel_shift_is_bit_exact_copy_and_periodic_wrap():
    import torch
    rng = np.random.default_rng(11)
    S, N = 64, 16
    scr = rng.standard_normal((S, S)).astype(np.float32)
    pupil = inputs.Pupil(N, 0.5, 4.0, 0.0)
    # wind 6 m/s along +x, -4 m/s along y, dt 0.25 s, pitch 0.5 m: 3 px and -2 px per step
    cfg = inputs.Config("shift", pupil, [], [inputs.Layer(S, 0.5, 0.0, 6.0, -4.0, 1.0, scr)],
                        [inputs.Source(0.0, 0.0, math.inf, 500e-9, -1)], 1, dt_s=0.25)
    inputs.fill_masks(cfg)
    geo = _geo(cfg, 1)
    ph = geo.trace_layers(1, 1, cfg.dt_s)
    torch.cuda.synchronize()
    got = geo.phase_view(ph, 0, 0).cpu().numpy()
    assert np.array_equal(got, scr[26:42, 21:37])
    # 40 steps: footprint has wrapped around the 64-px screen more than once; still equals the oracle
    ph = geo.trace_layers(40, 1, cfg.dt_s)
    ref = oracle.trace(cfg.layers, 0, 0, math.inf, 500e-9, 500e-9, N, 0.5, 40 * 0.25)
    assert np.array_equal(geo.phase_view(ph, 0, 0).cpu().numpy().astype(np.float64), ref)
    # non power-of-two screen with a footprint larger than the screen (wraps inside one call)
    scr2 = rng.standard_normal((48, 48)).astype(np.float32)
    cfg2 = inputs.Config("wrap", inputs.Pupil(100, 0.1, 5.0, 0.0), [],
                         [inputs.Layer(48, 0.13, 2000.0, 3.0, 1.0, 1.0, scr2)],
                         [inputs.Source(1e-4, -2e-4, 90e3, 589e-9, -1)], 1)
    inputs.fill_masks(cfg2)
    geo2 = _geo(cfg2, 1)
    ph2 = geo2.trace_layers(3, 2, cfg2.dt_s)
    torch.cuda.synchronize()
    for k in range(2):
        ref = oracle.trace(cfg2.layers, 1e-4, -2e-4, 90e3, 589e-9, 500e-9, 100, 0.1, (3 + k) * cfg2.dt_s)
        assert rel_l2(geo2.phase_view(ph2, 0, k).cpu().numpy(), ref) <= PHASE_TOL


def test_empty_and_error_cases():
    import torch
    from paper_1608_00386_b200 import binding
    cfg = inputs.make_config(0)
    geo = _geo(cfg, 1)
    # n_steps = 0 is a no-op
    geo.trace_layers(0, 0, cfg.dt_s, phase=torch.empty(1, device="cuda"))
    img, slp = geo.sh_images(0, None, 0, 0, cfg.dt_s)
    assert img.numel() == 0
    with pytest.raises(binding.AoError) as e:
        geo.sh_images(3, None, 0, 1, cfg.dt_s)
    assert e.value.status == 1
    with pytest.raises(binding.AoError) as e:
        geo.sh_images(0, None, 0, 1, cfg.dt_s, want_images=False, want_slopes=False)
    assert e.value.status == 1
    with pytest.raises(binding.AoError) as e:
        geo.psf(None, 0, 1, cfg.dt_s, psf=torch.empty(4, device="cuda"))   # no science direction
    assert e.value.status == 1
    # layer above the source altitude is skipped; no layers at all gives flat phase
    cfg2 = inputs.make_config(0, with_screens=False)
    cfg2.layers = []
    geo2 = _geo(cfg2, 1)
    ph = geo2.trace_layers(0, 1, cfg2.dt_s)
    torch.cuda.synchronize()
    assert float(ph.abs().max()) == 0.0
    assert geo2.launch_count() > 0 and geo.launch_count() == 0


def test_forward_host_matches_device_path():
    import torch
    cfg = inputs.make_config(3, n_sub=8, screen_n=512, n_steps=3)
    geo = _geo(cfg, 2)                                    # chunk of 2 steps < 3 steps: exercises chunking
    ref = oracle.forward(cfg, 0, 3, want_phase=False)
    sl = [torch.empty((3, len(cfg.sources_of_wfs(w)), 2, W.n_sub ** 2), dtype=torch.float32).pin_memory()
          for w, W in enumerate(cfg.wfs)]
    psf = torch.empty((len(cfg.science_sources()), cfg.psf_fft, cfg.psf_fft), dtype=torch.float32).pin_memory()
    scr = [torch.from_numpy(l.screen).pin_memory() for l in cfg.layers]
    for s in geo.screens:
        s.fill_(float("nan"))                              # the call must upload what it reads itself: anything it misses is NaN
    geo.forward_host(0, 3, cfg.dt_s, sl, psf, screens_host=scr)
    full = sum(l.n * l.n * 4 for l in cfg.layers)
    assert 0 < geo.last_h2d_bytes() < full                 # only the footprints' bounding box of every screen travels
    assert all(bool(torch.isfinite(t).all()) for t in sl) and bool(torch.isfinite(psf).all())
    for w in range(len(cfg.wfs)):
        for si, s in enumerate(cfg.sources_of_wfs(w)):
            for k in range(3):
                assert np.abs(sl[w][k, si].numpy() - ref["slopes"][s][k]).max() <= SLOPE_TOL
    for di, s in enumerate(cfg.science_sources()):
        assert rel_l2(psf[di].numpy(), ref["psf"][s]) <= IMAGE_TOL
    # far into the run the footprints have drifted across the periodic screen edge: the box is uploaded in pieces
    for s in geo.screens:
        s.fill_(float("nan"))
    ref2 = oracle.forward(cfg, 4000, 2, want_phase=False)
    geo.forward_host(4000, 2, cfg.dt_s, [t[:2] for t in sl], psf, screens_host=scr)
    for w in range(len(cfg.wfs)):
        for si, s in enumerate(cfg.sources_of_wfs(w)):
            for k in range(2):
                assert np.abs(sl[w][k, si].numpy() - ref2["slopes"][s][k]).max() <= SLOPE_TOL
    for di, s in enumerate(cfg.science_sources()):
        assert rel_l2(psf[di].numpy(), ref2["psf"][s]) <= IMAGE_TOL


@pytest.mark.parametrize("n_sub,psf_fft,n_steps", [(4, 64, 2), (20, None, 10), (40, None, 2), (20, 4096, 1), (80, None, 1)])
def test_big_fft_sizes_ngs_sensor_and_psf(n_sub, psf_fft, n_steps):
    """Two-pass register-resident FFT at every pass structure (16x4 .. 16x16x16): NGS sensor with
    FFT 64..1024 (2x2 subapertures, bin 8) and the science PSF with FFT 64..4096; the PSF long exposure
    is summed over more steps than one internal chunk holds (n_steps = 10)."""
    import torch
    cfg = inputs.make_config(4, n_sub=n_sub, screen_n=1024, n_steps=n_steps, lgs_fft=16, n_layers=2,
                             psf_fft=psf_fft)
    srcs = cfg.sources_of_wfs(1) + cfg.science_sources()
    ref = oracle.forward(cfg, 3, n_steps, want_phase=False, sources=srcs)
    geo = _geo(cfg, n_steps)
    img, slp = geo.sh_images(1, None, 3, n_steps, cfg.dt_s)
    torch.cuda.synchronize()
    check_wfs(cfg, geo, ref, 1, img, slp, n_steps, f"NGS fft {cfg.wfs[1].fft}")
    p = geo.psf(None, 3, n_steps, cfg.dt_s)
    p2 = geo.psf(None, 3, n_steps, cfg.dt_s, psf=p.clone(), accumulate=True)
    torch.cuda.synchronize()
    for di, s in enumerate(cfg.science_sources()):
        assert rel_l2(p[di].cpu().numpy(), ref["psf"][s]) <= IMAGE_TOL
        assert rel_l2(p2[di].cpu().numpy(), 2.0 * ref["psf"][s]) <= IMAGE_TOL
        assert abs(float(p[di].sum()) / n_steps - 1.0) < 1e-4          # Parseval: every PSF sums to 1


def _fused_vs_oracle(cfg, n_steps, step0):
    import torch
    ref = oracle.forward(cfg, step0, n_steps)
    geo = _geo(cfg, n_steps)
    img, slp = geo.sh_images(0, None, step0, n_steps, cfg.dt_s)
    torch.cuda.synchronize()
    return check_wfs(cfg, geo, ref, 0, img, slp, n_steps, cfg.name)


def test_fused_two_step_tiles_odd_counts_and_offsets():
    """The fused kernel pairs consecutive steps per CTA: odd step counts, odd first steps and a single
    step must give the same results as the oracle (the unpaired last step is computed but not stored)."""
    for n_steps, step0 in ((1, 0), (1, 7), (3, 1), (5, 498)):
        cfg = inputs.make_config(2, n_sub=9, screen_n=512, n_steps=n_steps)
        _fused_vs_oracle(cfg, n_steps, step0)


def test_fused_large_wind_shift_between_paired_steps():
    """Wind of 300 m/s: the two steps of a pair are 15 screen pixels apart, the staged box is their union
    (and wraps the periodic screen edge many times over 40 steps)."""
    cfg = inputs.make_config(2, n_sub=9, screen_n=512, n_steps=2)
    for i, lay in enumerate(cfg.layers):
        lay.wind_x_mps, lay.wind_y_mps = (300.0, -250.0) if i % 2 else (-280.0, 310.0)
    _fused_vs_oracle(cfg, 2, 39)


def test_low_altitude_source_takes_the_two_row_march():
    """A beacon at 30 km under 25 km of turbulence compresses the top layers to du = gamma d_s/d_l < 1/2,
    outside the three-term row march (1/2 <= du <= 1): the fused kernel and the tiled phase writer must switch to
    the two-row march (any du) and still match the oracle."""
    cfg = inputs.make_config(2, n_sub=9, screen_n=512, n_steps=2)
    for s in cfg.sources:
        s.altitude_m = 30e3
    _fused_vs_oracle(cfg, 2, 3)
    out = _run_all(cfg, 2, 3)
    ref = oracle.forward(cfg, 3, 2)
    _check_phase(cfg, out["geo"], out["phase"], ref, 2)


def test_forward_matches_separate_calls():
    """ao_forward (big-FFT sensors and PSF first, then the fused sensors, all on the caller's stream) gives
    the same slopes and long-exposure PSF as ao_sh_images per WFS plus ao_psf, bit for bit."""
    import torch
    cfg = inputs.make_config(3, n_sub=8, screen_n=512, n_steps=3)
    geo = _geo(cfg, 2)                                  # workspace of 2 steps: 3 steps run in two chunks
    ref_s = [geo.sh_images(w, None, 4, 3, cfg.dt_s, want_images=False)[1] for w in range(len(cfg.wfs))]
    ref_p = geo.psf(None, 4, 3, cfg.dt_s)
    torch.cuda.synchronize()
    got_s = [torch.full_like(r, float("nan")) for r in ref_s]
    got_p = torch.zeros_like(ref_p)
    for rep in range(2):                                # second call accumulates the PSF
        geo.forward(4, 3, cfg.dt_s, got_s, psf=got_p, accumulate=(rep == 1))
    torch.cuda.synchronize()
    for a, b in zip(got_s, ref_s):
        assert torch.equal(a, b)
    assert torch.allclose(got_p, 2.0 * ref_p, rtol=1e-6, atol=0.0)


def test_fft64_sensor_with_cropped_detector_window():
    """M = 64 sensors run one CTA per subaperture (both FFT passes in shared memory).  A detector that keeps the
    central 48 of 64 FFT pixels in 4 x 4 bins (k0 = 8, P = 12) exercises the window and binning arithmetic away from
    the c4 default (8 x 8 bins of the whole field); fine LGS grid: the phase comes from the quad row march."""
    cfg = inputs.make_config(4, n_sub=6, screen_n=1024, n_steps=3, lgs_fft=64)
    cfg.wfs[0].bin, cfg.wfs[0].n_pix = 4, 12
    ref = oracle.forward(cfg, 2, 3)
    geo = _geo(cfg, 3)
    import torch
    img, slp = geo.sh_images(0, None, 2, 3, cfg.dt_s)
    torch.cuda.synchronize()
    check_wfs(cfg, geo, ref, 0, img, slp, 3, cfg.name)


def _smooth_map(rng, N, rms):
    """Low-order random map (a few rad): bilinear upsampling of an 6 x 6 normal grid; harness data only."""
    g = rng.normal(size=(6, 6))
    x = np.linspace(0, 5, N)
    i0 = np.minimum(x.astype(int), 4); f = x - i0
    rows = g[i0] * (1 - f)[:, None] + g[i0 + 1] * f[:, None]
    m = rows[:, i0] * (1 - f)[None, :] + rows[:, i0 + 1] * f[None, :]
    return (rms * m).astype(np.float32)


def test_phase_maps_all_paths():
    """ao_set_phase_map (aberration maps summed to the open-loop wavefront): every phase producer
    -- tiled writer, fused kernel, big-FFT staging, PSF staging -- against the oracle; then clearing one map."""
    import torch
    cfg = inputs.make_config(3, n_sub=8, screen_n=512, n_steps=2)
    rng = np.random.default_rng(11)
    cfg.phase_maps = {s: _smooth_map(rng, cfg.grid_n(s), 2.0) for s in (0, 3, 6, 7, 9, 12)}   # LGS, NGS, science
    out, ref = _check_all(cfg, 2, step0=3)
    geo = out["geo"]
    # clear the map of LGS source 0: its slopes must go back to the map-free oracle values
    geo.set_phase_map(0, None)
    del cfg.phase_maps[0]
    ref0 = oracle.forward(cfg, 3, 2, sources=[0])
    img, slp = geo.sh_images(0, None, 3, 2, cfg.dt_s)
    torch.cuda.synchronize()
    d = np.abs(slp[:, 0].cpu().numpy() - ref0["slopes"][0]).max()
    assert d <= SLOPE_TOL, d


def test_phase_map_per_sample_trace_path_and_errors():
    """The per-sample kernel (screens whose side is not a multiple of 4 are outside the tile plan) adds the map too;
    bad source indices are rejected."""
    from paper_1608_00386_b200 import binding
    cfg = inputs.make_config(0)
    S = 254                                               # not a multiple of 4: k_trace path
    cfg.layers[0].screen = np.ascontiguousarray(cfg.layers[0].screen[:S, :S]); cfg.layers[0].n = S
    cfg.phase_maps = {0: _smooth_map(np.random.default_rng(2), cfg.grid_n(0), 1.0)}
    ref = oracle.forward(cfg, 0, 1)
    geo = _geo(cfg, 1)
    phase = geo.trace_layers(0, 1, cfg.dt_s)
    import torch
    torch.cuda.synchronize()
    _check_phase(cfg, geo, phase, ref, 1)
    with pytest.raises(binding.AoError):
        geo.set_phase_map(5, cfg.phase_maps[0])


def test_modes_to_map_and_closed_loop_residual():
    """ao_modes_to_map against the oracle contraction; then the residual-phase use: the map buffer is
    registered once with ao_set_phase_map and rewritten on the stream: the sensor sees open loop - DM shape."""
    import torch
    cfg = inputs.make_config(2, n_sub=9, screen_n=512, n_steps=2)
    geo = _geo(cfg, 2)
    rng = np.random.default_rng(21)
    N = cfg.grid_n(0)
    modes = np.ascontiguousarray(np.stack([_smooth_map(rng, N, 1.0) for _ in range(37)]))
    coeffs = rng.normal(size=37).astype(np.float32)
    d_modes, d_coeffs = torch.tensor(modes, device="cuda"), torch.tensor(coeffs, device="cuda")
    d_map = torch.full((N, N), float("nan"), dtype=torch.float32, device="cuda")
    geo.modes_to_map(d_modes, d_coeffs, -1.0, d_map)
    torch.cuda.synchronize()
    want = oracle.modes_to_map(modes, coeffs, -1.0)
    assert rel_l2(d_map.cpu().numpy(), want) <= 1e-6
    geo.set_phase_map(2, d_map)                               # LGS source 2 looks through the "mirror"
    for trial in range(2):                                    # new coefficients: same registered buffer, no re-registration
        c = rng.normal(size=37).astype(np.float32)
        geo.modes_to_map(d_modes, torch.tensor(c, device="cuda"), -1.0, d_map)
        img, slp = geo.sh_images(0, None, 7, 2, cfg.dt_s)
        torch.cuda.synchronize()
        cfg.phase_maps = {2: oracle.modes_to_map(modes, c, -1.0)}
        ref = oracle.forward(cfg, 7, 2, want_phase=False)
        check_wfs(cfg, geo, ref, 0, img, slp, 2, cfg.name + " residual")
    geo.modes_to_map(None, None, 1.0, d_map)                  # no modes: zero map
    torch.cuda.synchronize()
    assert float(d_map.abs().max()) == 0.0


def test_strehl_on_the_long_exposure_psf():
    """ao_strehl: peak of the long-exposure PSF over the diffraction-limited peak, against the oracle;
    a flat atmosphere gives Strehl 1 in every science direction."""
    import torch
    cfg = inputs.make_config(3, n_sub=8, screen_n=512, n_steps=3)
    geo = _geo(cfg, 3)
    psf = geo.psf(None, 0, 3, cfg.dt_s)
    got = geo.strehl(psf, 3).cpu().numpy()
    ref = oracle.forward(cfg, 0, 3, want_phase=False, want_wfs=False)
    want = np.array([oracle.strehl(ref["psf"][s], cfg.pupil.amp, 3) for s in cfg.science_sources()])
    assert got.shape == want.shape and np.abs(got - want).max() <= 1e-5 * max(1.0, np.abs(want).max())
    assert (want < 0.9).all()                                  # the turbulence does degrade the image
    for lay in cfg.layers:
        lay.screen = np.zeros_like(lay.screen)
    flat = _geo(cfg, 1)
    s1 = flat.strehl(flat.psf(None, 0, 1, cfg.dt_s), 1).cpu().numpy()
    assert np.abs(s1 - 1.0).max() <= 1e-5
    from paper_1608_00386_b200 import binding
    with pytest.raises(binding.AoError):
        flat.strehl(psf, 0)                                    # n_exposures must be positive


def test_marechal_strehl_on_traced_phase():
    """ao_strehl_marechal on the ao_trace_layers buffer against the oracle, with a residual-phase map on
    one science direction; open-loop phase variances are hundreds of rad^2, so compare the exponent too."""
    import torch
    cfg = inputs.make_config(3, n_sub=8, screen_n=512, n_steps=2)
    sci = cfg.science_sources()
    for lay in cfg.layers:                                   # weak turbulence: Strehl values of order 0.1 - 0.9
        lay.screen = (0.3 * lay.screen).astype(np.float32)
    cfg.phase_maps = {sci[1]: _smooth_map(np.random.default_rng(3), cfg.grid_n(sci[1]), 0.3)}
    geo = _geo(cfg, 2)
    phase = geo.trace_layers(5, 2, cfg.dt_s)
    got = geo.strehl_marechal(phase, 2).cpu().numpy().astype(np.float64)
    ref = oracle.forward(cfg, 5, 2, want_wfs=False, want_psf=False, sources=sci)
    want = np.array([[oracle.strehl_marechal(ref["phase"][s][k], cfg.pupil.amp) for s in sci] for k in range(2)])
    assert got.shape == want.shape
    assert np.abs(got - want).max() <= 1e-5
    assert (want > 0.01).all() and (want < 0.99).all(), want       # neither saturated nor trivial


@pytest.mark.parametrize("M", [16, 32, 64])
def test_lgs_spot_elongation_all_paths(M):
    """NEXT-3 (reading O9): extended sodium layer with a time-varying profile and side launch.  The fused
    kernel (M = 16, 32: k_fused<..., ELONG>), the phase-buffer path and M = 64 (k_sh_generic) against the oracle, over
    steps that wrap the profile table; then the point beacon again after clearing the profile."""
    import torch
    cfg = inputs.make_config(4, n_sub=10, screen_n=1024, n_steps=3, lgs_fft=M, n_layers=6)
    cfg.sources = cfg.sources[:6]; cfg.wfs = cfg.wfs[:1]; cfg.psf_fft = 0
    cfg.sodium = inputs.sodium_profile(cfg, n_z=5, n_t=4, launch="side", fwhm_m=2e3)
    ref = oracle.forward(cfg, 6, 3)
    geo = _geo(cfg, 3)
    img, slp = geo.sh_images(0, None, 6, 3, cfg.dt_s)
    phase = geo.trace_layers(6, 3, cfg.dt_s)
    img_p, slp_p = geo.sh_images(0, phase, 6, 3, cfg.dt_s)
    torch.cuda.synchronize()
    a = check_wfs(cfg, geo, ref, 0, img, slp, 3, f"elongation M={M}, phase_dev = NULL")
    b = check_wfs(cfg, geo, ref, 0, img_p, slp_p, 3, f"elongation M={M}, phase buffer")
    from tests.parity_util import report
    report(f"elongation_M{M}", images_rel_l2=max(a[0], b[0]), slopes_max_abs=max(a[1], b[1]), per_subap_rel_l2=max(a[2], b[2]))
    # the spots are longer than a point beacon's: the brightest pixel drops
    cfg.sodium = None
    point = oracle.forward(cfg, 6, 1, want_phase=False)
    assert ref["images"][0][0].max() < point["images"][0][0].max()
    geo.set_sodium(None)
    img0, slp0 = geo.sh_images(0, None, 6, 1, cfg.dt_s)
    torch.cuda.synchronize()
    check_wfs(cfg, geo, point, 0, img0, slp0, 1, "point beacon after clearing the profile")


def test_lgs_spot_elongation_with_noise_and_errors():
    """Detector noise on elongated spots through the fused kernel (k_fused<32, NOISE, ..., ELONG>); ao_set_sodium rejects
    sensors of natural stars and big-FFT sensors."""
    import torch
    from paper_1608_00386_b200 import binding
    cfg = inputs.make_config(2, n_sub=9, screen_n=512, n_steps=1)
    cfg.sodium = inputs.sodium_profile(cfg, n_z=3, n_t=1, fwhm_m=1.5e3)
    ref = oracle.forward(cfg, 4, 1, want_phase=False, noise_on=True)
    geo = _geo(cfg, 1)
    noisy, slopes = geo.sh_images(0, None, 4, 1, cfg.dt_s, noise=cfg.noise)
    torch.cuda.synchronize()
    tot = bad = 0
    for si, s in enumerate(cfg.sources_of_wfs(0)):
        same = np.abs(noisy[0, si].cpu().numpy().astype(np.float64) - ref["noisy"][s][0]) < 0.5
        tot += same.size; bad += int((~same).sum())
        ok = same.reshape(same.shape[0], -1).all(axis=1)
        d = np.abs(slopes[0, si].cpu().numpy().astype(np.float64) - ref["slopes"][s][0])
        assert d[:, ok].max() <= SLOPE_TOL
    assert bad <= max(1, int(1e-5 * tot))
    c3 = inputs.make_config(3, n_sub=8, screen_n=512, n_steps=1)
    g3 = _geo(c3, 1)
    na = inputs.sodium_profile(c3, wfs_index=1, n_z=3, n_t=1)
    with pytest.raises(binding.AoError):
        g3.set_sodium(na)                                    # NGS sensor: sources at infinity / fft > 64


@pytest.mark.parametrize("n_sub,n_steps", [(8, 3), (20, 2)])
def test_polychromatic_psf_against_the_oracle(n_sub, n_steps):
    """NEXT-4 (reading O8): ao_psf_poly over a three-wavelength band (chirp-z scaled DFTs on the pixel grid
    of the directions' own wavelength) against the oracle's F E F^T definition; from a phase buffer and with the library's
    own ray-trace, accumulating, through ao_forward, and one wavelength = ao_psf."""
    import torch
    cfg = inputs.make_config(3, n_sub=n_sub, screen_n=512, n_steps=n_steps)
    cfg.sources = cfg.sources[:9] + cfg.sources[9:12]                 # three science directions are enough
    cfg.psf_band = ([1.9e-6, 2.2e-6, 2.45e-6], [0.25, 0.45, 0.30])
    sci = cfg.science_sources()
    ref = oracle.forward(cfg, 2, n_steps, want_phase=False, want_wfs=False, sources=sci)
    geo = _geo(cfg, n_steps)
    p = geo.psf_poly(None, 2, n_steps, cfg.dt_s)
    phase = geo.trace_layers(2, n_steps, cfg.dt_s)
    p2 = geo.psf_poly(phase, 2, n_steps, cfg.dt_s, psf=p.clone(), accumulate=True)
    torch.cuda.synchronize()
    worst = 0.0
    for di, s in enumerate(sci):
        worst = max(worst, rel_l2(p[di].cpu().numpy(), ref["psf"][s]), rel_l2(p2[di].cpu().numpy(), 2.0 * ref["psf"][s]))
    assert worst <= IMAGE_TOL, worst
    from tests.parity_util import report
    report(f"psf_poly_nsub{n_sub}", psf_rel_l2=worst)
    # ao_forward uses the band while it is set
    sl = [torch.empty((n_steps, len(cfg.sources_of_wfs(w)), 2, W.n_sub ** 2), dtype=torch.float32, device="cuda")
          for w, W in enumerate(cfg.wfs)]
    pf = torch.zeros_like(p)
    geo.forward(2, n_steps, cfg.dt_s, sl, psf=pf)
    torch.cuda.synchronize()
    assert torch.allclose(pf, p, rtol=1e-6, atol=0.0)
    # a band of the directions' own wavelength alone is the monochromatic PSF (two different transforms: chirp-z, FFT)
    geo.set_psf_band([2.2e-6], [1.0])
    mono = geo.psf(None, 2, n_steps, cfg.dt_s)
    one = geo.psf_poly(None, 2, n_steps, cfg.dt_s)
    torch.cuda.synchronize()
    for di in range(len(sci)):
        assert rel_l2(one[di].cpu().numpy(), mono[di].cpu().numpy().astype(np.float64)) <= IMAGE_TOL
    geo.set_psf_band(None)
    from paper_1608_00386_b200 import binding
    with pytest.raises(binding.AoError):
        geo.psf_poly(None, 2, 1, cfg.dt_s)


def test_fused64_odd_counts_phase_maps_and_noise():
    """k_fused64 (M = 64, n = 32: the tile marched twice per subaperture row): odd step counts and odd first steps, a static
    phase map on two of the six LGS (the kernel reads sp.map), and detector noise through the fused kernel
    (k_fused64<..., NOISE>) under the protocol of reading O5."""
    import torch
    for n_steps, step0 in ((1, 7), (3, 498)):
        cfg = inputs.make_config(4, n_sub=6, screen_n=1024, n_steps=n_steps, lgs_fft=64, n_layers=7)
        cfg.sources = cfg.sources[:6]; cfg.wfs = cfg.wfs[:1]; cfg.psf_fft = 0
        rng = np.random.default_rng(5)
        cfg.phase_maps = {s: _smooth_map(rng, cfg.grid_n(s), 1.5) for s in (1, 4)}
        ref = oracle.forward(cfg, step0, n_steps, want_phase=False)
        geo = _geo(cfg, n_steps)
        img, slp = geo.sh_images(0, None, step0, n_steps, cfg.dt_s)
        torch.cuda.synchronize()
        check_wfs(cfg, geo, ref, 0, img, slp, n_steps, f"k_fused64 {n_steps} steps from {step0}")
    cfg.noise = inputs.Noise(seed=99, photons_per_subap=4000.0, read_noise_e=2.0)
    refn = oracle.forward(cfg, 498, 3, want_phase=False, noise_on=True)
    noisy, slopes = geo.sh_images(0, None, 498, 3, cfg.dt_s, noise=cfg.noise)
    torch.cuda.synchronize()
    tot = bad = 0
    for si, s in enumerate(cfg.sources_of_wfs(0)):
        for k in range(3):
            same = np.abs(noisy[k, si].cpu().numpy().astype(np.float64) - refn["noisy"][s][k]) < 0.5
            tot += same.size; bad += int((~same).sum())
            ok = same.reshape(same.shape[0], -1).all(axis=1)
            d = np.abs(slopes[k, si].cpu().numpy().astype(np.float64) - refn["slopes"][s][k])
            assert d[:, ok].max() <= SLOPE_TOL
    assert bad <= max(1, int(1e-5 * tot)), (bad, tot)
