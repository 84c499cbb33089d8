"""Pins for the FP64 oracle (oracle/ao_oracle.c) against things other than itself:
closed forms, brute force, library routines, invariants and the values printed in
SURVEY.md §8(c) (tests/golden/sh_closed_form.txt).  CPU only.

Every pin is chosen so that a plausible mistake (dropped term, wrong sign or index,
transposed operand, wrong centring, wrong normalisation) fails at least one of them.
"""
import ctypes as C
import math
import os

import numpy as np
import pytest

import oracle
from paper_1608_00386_b200 import inputs
from tests.golden_io import load as load_golden

GOLD = load_golden()
RNG = np.random.default_rng(20160800386)


# ----------------------------------------------------------------------------- helpers
def dirichlet_binned(n, M, beta, P, alpha):
    """1-D closed form: |sum_{a<n} exp(i a psi)|^2 = sin^2(n psi/2)/sin^2(psi/2), psi = alpha-2 pi nu/M,
    nu = k-(M-1)/2, normalised by M n (Parseval) and binned.  Independent of the oracle."""
    nu = np.arange(M) - (M - 1) / 2.0
    psi = alpha - 2.0 * np.pi * nu / M
    s = np.sin(psi / 2.0)
    with np.errstate(all="ignore"):
        D = np.where(np.abs(s) < 1e-13, float(n * n), np.sin(n * psi / 2.0) ** 2 / s ** 2)
    prof = D / (M * n)
    k0 = (M - beta * P) // 2
    return prof[k0:k0 + beta * P].reshape(P, beta).sum(1)


def one_subap(phase_block, n, M, beta, P, amp=None):
    amp = np.ones((n, n), np.float32) if amp is None else amp
    img, valid = oracle.sh_images(phase_block, amp, 1, n, M, beta, P, 0.0)
    return img[0], valid[0]


def make_layer(screen, pitch=0.1, h=0.0, wx=0.0, wy=0.0):
    return inputs.Layer(screen.shape[0], pitch, h, wx, wy, 1.0, screen.astype(np.float32))


# ----------------------------------------------------------------------------- DFT core
def brute_dft2(block, M, c):
    """O(N^4) definition: out[k][m] = sum_ab in[a][b] exp(-2 pi i ((k-c) a + (m-c) b)/M), python loops."""
    n = block.shape[0]
    out = np.zeros((M, M), complex)
    for k in range(M):
        for m in range(M):
            acc = 0j
            for a in range(n):
                for b in range(n):
                    acc += block[a, b] * np.exp(-2j * np.pi * ((k - c) * a + (m - c) * b) / M)
            out[k, m] = acc
    return out


@pytest.mark.parametrize("half", [0, 1])
@pytest.mark.parametrize("method", [0, 1])
def test_dft_matches_brute_force_8x8(half, method):
    blk = RNG.standard_normal((8, 8)) + 1j * RNG.standard_normal((8, 8))
    ref = brute_dft2(blk, 8, 3.5 if half else 4.0)
    got = oracle.cdft2(blk, 8, bool(half), method)
    assert np.abs(got - ref).max() <= 1e-13 * np.abs(ref).max() * 8


def test_dft_zero_padded_brute_force_nonsquare_sizes():
    # n < M (zero padding) and a non power of two M=12 (direct method only)
    blk = RNG.standard_normal((5, 5)) + 1j * RNG.standard_normal((5, 5))
    for half in (0, 1):
        ref = brute_dft2(blk, 12, 5.5 if half else 6.0)
        got = oracle.cdft2(blk, 12, bool(half), 0)
        assert np.abs(got - ref).max() < 1e-12


def test_pixel_centred_dft_is_numpy_fftshift():
    # nu_k = k - M/2  <=>  fftshift(fft2(zero-padded block)): an independent library routine
    n, M = 12, 32
    blk = RNG.standard_normal((n, n)) + 1j * RNG.standard_normal((n, n))
    pad = np.zeros((M, M), complex); pad[:n, :n] = blk
    ref = np.fft.fftshift(np.fft.fft2(pad))
    for method in (0, 1):
        got = oracle.cdft2(blk, M, False, method)
        assert np.abs(got - ref).max() < 1e-11


def test_half_pixel_dft_is_numpy_fft_of_ramped_input():
    # nu_k = k-(M-1)/2: exp(-2 pi i nu a/M) = exp(-2 pi i k a/M) exp(+i pi (M-1) a/M)
    n, M = 12, 24
    blk = RNG.standard_normal((n, n)) + 1j * RNG.standard_normal((n, n))
    a = np.arange(M)
    ramp = np.exp(1j * np.pi * (M - 1) * a / M)
    pad = np.zeros((M, M), complex); pad[:n, :n] = blk
    ref = np.fft.fft2(pad * ramp[:, None] * ramp[None, :])
    got = oracle.cdft2(blk, M, True, 0)
    assert np.abs(got - ref).max() < 1e-11


@pytest.mark.parametrize("n,M", [(32, 64), (48, 128), (64, 64)])
def test_radix2_fft_matches_direct_dft(n, M):
    blk = RNG.standard_normal((n, n)) + 1j * RNG.standard_normal((n, n))
    for half in (False, True):
        d = oracle.cdft2(blk, M, half, 0)
        f = oracle.cdft2(blk, M, half, 1)
        assert np.abs(d - f).max() <= 1e-12 * np.abs(d).max()


def test_dft_linearity_and_parseval():
    n, M = 8, 16
    x = RNG.standard_normal((n, n)) + 1j * RNG.standard_normal((n, n))
    y = RNG.standard_normal((n, n)) + 1j * RNG.standard_normal((n, n))
    for half in (False, True):
        fx, fy = oracle.cdft2(x, M, half, 0), oracle.cdft2(y, M, half, 0)
        fxy = oracle.cdft2(2.0 * x - 3j * y, M, half, 0)
        assert np.abs(fxy - (2.0 * fx - 3j * fy)).max() < 1e-12
        assert abs((np.abs(fx) ** 2).sum() - M * M * (np.abs(x) ** 2).sum()) < 1e-9


def test_dft_row_column_orientation():
    # a delta at in[a0][b0] must give exp(-2 pi i (nu_k a0 + nu_m b0)/M): catches transposed operands
    n, M = 8, 16
    blk = np.zeros((n, n), complex); blk[3, 1] = 1.0
    got = oracle.cdft2(blk, M, True, 0)
    nu = np.arange(M) - (M - 1) / 2
    ref = np.exp(-2j * np.pi * (nu[:, None] * 3 + nu[None, :] * 1) / M)
    assert np.abs(got - ref).max() < 1e-13


# ----------------------------------------------------------------------------- SH images
@pytest.mark.parametrize("key", list(GOLD["profile"].keys()))
def test_flat_subaperture_profile_matches_golden_and_dirichlet(key):
    n, M, beta, P = key
    img, _ = one_subap(np.zeros((n, n)), n, M, beta, P)
    prof = np.array(GOLD["profile"][key])
    full = np.concatenate([prof, prof[::-1]])
    # 2-D image = outer product of the 1-D profiles (separable flat square subaperture: "sinc^2" pin)
    assert np.abs(img - np.outer(full, full)).max() < 2e-12
    d = dirichlet_binned(n, M, beta, P, 0.0)
    assert np.abs(img - np.outer(d, d)).max() < 1e-14
    assert abs(img.sum() - 1.0) < 1e-13


def test_c0_centre_pixels_value():
    img, _ = one_subap(np.zeros((8, 8)), 8, 16, 2, 8)
    assert abs(img[3, 3] - 0.452945956815 ** 2) < 1e-11      # = 0.205160
    assert abs(img[3, 3] - 0.205160) < 1e-6
    assert abs(img[3, 3] - img[4, 4]) < 1e-16 and abs(img[3, 4] - img[4, 3]) < 1e-16


@pytest.mark.parametrize("n,M,beta,P", [(8, 16, 2, 8), (12, 24, 4, 6), (16, 32, 4, 8), (32, 64, 8, 8)])
def test_flat_gives_zero_slopes(n, M, beta, P):
    img, valid = one_subap(np.zeros((n, n)), n, M, beta, P)
    s = oracle.centroids(img[None], np.array([valid]))
    assert np.abs(s).max() < 1e-15


def test_piston_invariance():
    n, M, beta, P = 16, 32, 4, 8
    ph = RNG.standard_normal((n, n)) * 2.0
    a, _ = one_subap(ph, n, M, beta, P)
    b, _ = one_subap(ph + 12.345, n, M, beta, P)
    assert np.abs(a - b).max() < 1e-13


@pytest.mark.parametrize("entry", GOLD["cog"])
def test_tilt_cog_matches_golden(entry):
    (n, M, beta, P), t, cog = entry
    alpha = 2.0 * np.pi * t / M
    b = np.arange(n)
    # x tilt: phase grows along the column index b -> spot moves to +column -> s_x > 0, s_y = 0
    img, valid = one_subap(np.tile(alpha * b, (n, 1)), n, M, beta, P)
    s = oracle.centroids(img[None], np.array([valid]))
    assert abs(s[0, 0] - cog) < 2e-12
    assert abs(s[1, 0]) < 1e-14
    # y tilt: phase grows along the row index a -> s_y = cog, s_x = 0
    img, valid = one_subap(np.tile(alpha * b[:, None], (1, n)), n, M, beta, P)
    s = oracle.centroids(img[None], np.array([valid]))
    assert abs(s[1, 0] - cog) < 2e-12 and abs(s[0, 0]) < 1e-14
    # and against the Dirichlet closed form evaluated here
    d = dirichlet_binned(n, M, beta, P, alpha)
    assert abs((d * (np.arange(P) - (P - 1) / 2)).sum() / d.sum() - cog) < 2e-12


def test_integer_tilt_is_exact_circular_shift():
    # alpha = 2 pi t / M, integer t: the unbinned image (beta = 1, P = M) shifts circularly by t
    n, M = 8, 16
    base, _ = one_subap(np.zeros((n, n)), n, M, 1, M)
    for t in (1, 3, -2):
        ph = np.tile(2 * np.pi * t / M * np.arange(n), (n, 1))
        img, _ = one_subap(ph, n, M, 1, M)
        assert np.abs(img - np.roll(base, t, axis=1)).max() < 1e-13
    # t a multiple of beta: the binned image shifts by whole detector pixels
    n, M, beta, P = 16, 32, 4, 8
    base, _ = one_subap(np.zeros((n, n)), n, M, beta, P)
    ph = np.tile(2 * np.pi * beta / M * np.arange(n)[:, None], (1, n))
    img, _ = one_subap(ph, n, M, beta, P)
    assert np.abs(img - np.roll(base, 1, axis=0)).max() < 1e-13


def test_partial_illumination_energy_and_validity():
    n, M, beta, P = 8, 16, 2, 8
    amp = np.ones((n, n), np.float32); amp[:, :3] = 0.0           # 5/8 lit
    ph = RNG.standard_normal((n, n))
    img, valid = oracle.sh_images(ph, amp, 1, n, M, beta, P, 0.5)
    assert valid[0] == 1 and abs(img.sum() - 5.0 / 8.0) < 1e-13     # Parseval: sum = lit fraction
    amp[:, :5] = 0.0                                               # 3/8 lit < 0.5 -> invalid -> zeros
    img, valid = oracle.sh_images(ph, amp, 1, n, M, beta, P, 0.5)
    assert valid[0] == 0 and np.all(img == 0.0)
    assert np.all(oracle.centroids(img, valid) == 0.0)


def test_cropped_window_is_central():
    # beta*P < M: the detector is the central window of the binned full field
    n, M, beta = 8, 16, 2
    ph = RNG.standard_normal((n, n))
    full, _ = one_subap(ph, n, M, beta, 8)
    crop, _ = one_subap(ph, n, M, beta, 4)
    assert np.abs(crop - full[2:6, 2:6]).max() < 1e-15


def test_subaperture_blocks_are_indexed_row_major():
    # a 2x2 WFS: subaperture (p, q) must use rows p*n.., columns q*n.. of the phase
    n, M, beta, P = 8, 16, 2, 8
    ph = RNG.standard_normal((2 * n, 2 * n))
    amp = np.ones((2 * n, 2 * n), np.float32)
    img, _ = oracle.sh_images(ph, amp, 2, n, M, beta, P, 0.5)
    for p in range(2):
        for q in range(2):
            one, _ = one_subap(ph[p * n:(p + 1) * n, q * n:(q + 1) * n], n, M, beta, P)
            assert np.abs(img[p * 2 + q] - one).max() < 1e-15


def test_mask_counts_match_survey():
    c = GOLD["count"]
    cfg = inputs.make_config(0, with_screens=False)
    W = cfg.wfs[0]
    assert int(cfg.pupil.amp.sum()) == c["c0"]["lit"]
    _, valid = oracle.sh_images(np.zeros((80, 80)), W.amp, 10, 8, 16, 2, 8, 0.5)
    assert int(valid.sum()) == c["c0"]["valid"]
    blocks = W.amp.reshape(10, 8, 10, 8).transpose(0, 2, 1, 3).reshape(100, 64)
    assert int((blocks.sum(1) == 64).sum()) == c["c0"]["fully_lit"]
    m960 = inputs.annulus_mask(960, 0.04, 19.2, 5.5)
    assert int(m960.sum()) == c["elt960"]["lit"]
    b = m960.reshape(80, 12, 80, 12).transpose(0, 2, 1, 3).reshape(6400, 144).sum(1)
    assert int((b >= 72).sum()) == c["elt960"]["valid"] and int((b == 144).sum()) == c["elt960"]["fully_lit"]
    m1280 = inputs.annulus_mask(1280, 0.03, 19.2, 5.5)
    assert int(m1280.sum()) == c["elt1280"]["lit"]
    b = m1280.reshape(80, 16, 80, 16).transpose(0, 2, 1, 3).reshape(6400, 256).sum(1)
    assert int((b >= 128).sum()) == c["elt1280"]["valid"]


# ----------------------------------------------------------------------------- centroid
def test_centroid_of_delta_and_sign_convention():
    P = 8
    img = np.zeros((3, P, P))
    img[0, 2, 6] = 5.0          # row 2, column 6
    img[1, :, :] = 1.0          # uniform -> 0
    img[2, 7, 0] = 1.0; img[2, 0, 7] = 1.0
    s = oracle.centroids(img)
    assert s.shape == (2, 3)
    assert s[0, 0] == 6 - 3.5 and s[1, 0] == 2 - 3.5
    assert s[0, 1] == 0.0 and s[1, 1] == 0.0
    assert s[0, 2] == 0.0 and s[1, 2] == 0.0
    assert np.all(oracle.centroids(np.zeros((1, P, P))) == 0.0)     # |sum| < 1e-12 -> 0


# ----------------------------------------------------------------------------- trace
def test_bilinear_of_linear_screen_is_exact():
    S, N, d = 64, 16, 0.1
    c0, cr, cc = 1.5, 0.25, -0.125
    lay = make_layer(inputs.linear_screen(S, c0, cr, cc), pitch=0.1, h=1000.0, wx=3.0, wy=-2.0)
    th = (2e-4, -1e-4); t = 0.05; H = 90e3; lam = 589e-9
    ph = oracle.trace([lay], th[0], th[1], H, lam, 500e-9, N, d, t)
    g = 1 - 1000.0 / H
    x = (np.arange(N) - (N - 1) / 2) * d
    u = (g * x + 1000.0 * th[0] - 3.0 * t) / 0.1 + (S - 1) / 2
    v = (g * x + 1000.0 * th[1] + 2.0 * t) / 0.1 + (S - 1) / 2
    ref = (c0 + cr * v[:, None] + cc * u[None, :]) * 500e-9 / lam
    assert np.abs(ph - ref).max() < 1e-12


def test_integer_pixel_shift_is_exact_subarray_copy():
    S, N = 64, 16
    scr = RNG.standard_normal((S, S)).astype(np.float32)
    # v t / d = 3 px in x, -2 px in y; gamma = 1, theta = 0, lambda = lambda_ref, pitch ratio 1
    lay = make_layer(scr, pitch=0.5, wx=3 * 0.5 / 0.25, wy=-2 * 0.5 / 0.25)
    ph = oracle.trace([lay], 0, 0, math.inf, 500e-9, 500e-9, N, 0.5, 0.25)
    j0 = (S - 1) // 2 - (N - 1) // 2 - 3        # u = j - 7.5 - 3 + 31.5 = j + 21
    i0 = (S - 1) // 2 - (N - 1) // 2 + 2
    assert np.array_equal(ph, scr[i0:i0 + N, j0:j0 + N].astype(np.float64))


def test_half_pixel_shift_is_mean_of_neighbours_and_wind_sign():
    S, N = 32, 8
    scr = RNG.standard_normal((S, S)).astype(np.float32)
    lay = make_layer(scr, pitch=1.0, wx=0.5, wy=0.0)          # screen moves +x by 0.5 px at t = 1
    ph = oracle.trace([lay], 0, 0, math.inf, 500e-9, 500e-9, N, 1.0, 1.0)
    # pupil samples screen coordinate x - v t: u = j - 3.5 - 0.5 + 15.5 = j + 11.5
    ref = 0.5 * (scr[12:20, 11:19].astype(np.float64) + scr[12:20, 12:20])
    assert np.abs(ph - ref).max() < 1e-15


def test_off_axis_source_shifts_by_h_theta():
    S, N = 64, 8
    scr = RNG.standard_normal((S, S)).astype(np.float32)
    h, dl = 10000.0, 0.25
    lay = make_layer(scr, pitch=dl, h=h)
    base = oracle.trace([lay], 0, 0, math.inf, 500e-9, 500e-9, N, dl, 0.0)
    # theta_x = 2^-15 rad with h d_l^-1 = 40000: shift = 40000/32768 px is not integer; use exact one:
    ph = oracle.trace([lay], dl / h, 0, math.inf, 500e-9, 500e-9, N + 1, dl, 0.0)
    big = oracle.trace([lay], 0, 0, math.inf, 500e-9, 500e-9, N + 1, dl, 0.0)
    # +theta displaces the footprint by +h theta = +1 px along x
    assert np.abs(ph[:, :-1] - big[:, 1:]).max() < 1e-9
    phy = oracle.trace([lay], 0, dl / h, math.inf, 500e-9, 500e-9, N + 1, dl, 0.0)
    assert np.abs(phy[:-1, :] - big[1:, :]).max() < 1e-9
    assert base.shape == (N, N)


def test_cone_effect_scales_gradient():
    # linear screen, LGS at H: recovered gradient = c * gamma * d_s / d_l per sample
    S, N = 128, 16
    cc = 0.25          # exactly representable in fp32 for all j < S
    lay = make_layer(inputs.linear_screen(S, 0.0, 0.0, cc), pitch=0.04, h=15000.0)
    H = 90e3
    ph = oracle.trace([lay], 0, 0, H, 500e-9, 500e-9, N, 0.03, 0.0)
    grad = np.diff(ph, axis=1)
    assert np.abs(grad - cc * (1 - 15000.0 / H) * 0.03 / 0.04).max() < 1e-12
    assert np.abs(np.diff(ph, axis=0)).max() < 1e-12
    # layer at/above the source altitude is skipped
    top = make_layer(inputs.linear_screen(S, 7.0, 0.0, 0.0), pitch=0.04, h=H)
    ph2 = oracle.trace([lay, top], 0, 0, H, 500e-9, 500e-9, N, 0.03, 0.0)
    assert np.array_equal(ph, ph2)


def test_periodicity_wavelength_scaling_and_layer_sum():
    S, N = 32, 12
    a = make_layer(RNG.standard_normal((S, S)), pitch=0.1, h=0.0, wx=1.0, wy=2.0)
    b = make_layer(RNG.standard_normal((S, S)), pitch=0.1, h=5000.0, wx=-3.0, wy=0.5)
    args = (1e-5, -2e-5, math.inf)
    p0 = oracle.trace([a, b], *args, 500e-9, 500e-9, N, 0.1, 0.37)
    # shifting by exactly S pixels (t -> t + S d / v for a single layer) returns the same phase
    pa = oracle.trace([a], *args, 500e-9, 500e-9, N, 0.1, 0.37)
    pa2 = oracle.trace([a], *args, 500e-9, 500e-9, N, 0.1, 0.37 + S * 0.1 / 1.0)
    assert np.abs(pa - pa2).max() < 1e-9
    # also wraps across the edge: a sample footprint larger than the screen still works
    wide = oracle.trace([a], 0, 0, math.inf, 500e-9, 500e-9, 2 * S, 0.1, 0.0)
    assert np.abs(wide[:S, :S] - wide[S:, S:]).max() < 1e-9
    # lambda scaling and additivity over layers
    p1 = oracle.trace([a, b], *args, 2.2e-6, 500e-9, N, 0.1, 0.37)
    assert np.abs(p1 - p0 * (500e-9 / 2.2e-6)).max() < 1e-13
    pb = oracle.trace([b], *args, 500e-9, 500e-9, N, 0.1, 0.37)
    assert np.abs(p0 - (pa + pb)).max() < 1e-13


def test_trace_matches_scipy_map_coordinates():
    # an independent library routine: order-1 spline interpolation with periodic ('grid-wrap') boundary
    from scipy.ndimage import map_coordinates
    S, N, d, dl = 48, 20, 0.03, 0.04
    scr = RNG.standard_normal((S, S)).astype(np.float32)
    lay = make_layer(scr, pitch=dl, h=8000.0, wx=7.0, wy=-11.0)
    H, thx, thy, t = 90e3, 1.5e-4, -0.7e-4, 0.123
    ph = oracle.trace([lay], thx, thy, H, 500e-9, 500e-9, N, d, t)
    g = 1 - 8000.0 / H
    x = (np.arange(N) - (N - 1) / 2) * d
    u = (g * x + 8000.0 * thx - 7.0 * t) / dl + (S - 1) / 2
    v = (g * x + 8000.0 * thy + 11.0 * t) / dl + (S - 1) / 2
    vv, uu = np.meshgrid(v, u, indexing="ij")
    ref = map_coordinates(scr.astype(np.float64), [vv, uu], order=1, mode="grid-wrap")
    assert np.abs(ph - ref).max() < 1e-12


def test_end_to_end_linear_screen_gives_closed_form_slopes():
    # linear screen of g rad/px through O2 -> alpha = g gamma (d_s/d_l)(lambda_ref/lambda) -> CoG closed form
    n_sub, n, M, beta, P = 4, 16, 32, 4, 8
    N = n_sub * n
    g_px = 0.1875      # exactly representable in fp32 for all j < S
    S = 256
    lay = make_layer(inputs.linear_screen(S, 0.0, 0.0, g_px), pitch=0.04, h=10000.0)
    H, lam = 90e3, 589e-9
    d_s = 0.03
    ph = oracle.trace([lay], 0, 0, H, lam, 500e-9, N, d_s, 0.0)
    img, valid = oracle.sh_images(ph, np.ones((N, N), np.float32), n_sub, n, M, beta, P, 0.5)
    s = oracle.centroids(img, valid)
    alpha = g_px * (1 - 10000.0 / H) * d_s / 0.04 * 500e-9 / lam
    d = dirichlet_binned(n, M, beta, P, alpha)
    cog = (d * (np.arange(P) - (P - 1) / 2)).sum() / d.sum()
    assert np.abs(s[0] - cog).max() < 1e-11 and np.abs(s[1]).max() < 1e-11


# ----------------------------------------------------------------------------- PSF
def test_psf_square_flat_pupil_is_dirichlet_product():
    N, M = 12, 32
    p = oracle.psf(np.zeros((N, N)), np.ones((N, N), np.float32), M)
    nu = np.arange(M) - M / 2
    psi = -2 * np.pi * nu / M
    s = np.sin(psi / 2)
    with np.errstate(all="ignore"):
        D = np.where(np.abs(s) < 1e-13, float(N * N), np.sin(N * psi / 2) ** 2 / s ** 2) / (M * N)
    assert np.abs(p - np.outer(D, D)).max() < 1e-14
    assert np.unravel_index(np.argmax(p), p.shape) == (M // 2, M // 2)
    assert abs(p.sum() - 1.0) < 1e-13


def test_psf_circular_flat_pupil_peak_symmetry_shift_and_accumulate():
    N, M = 48, 128
    amp = inputs.annulus_mask(N, 0.04, N * 0.02, 0.2)
    lit = float(amp.sum())
    p = oracle.psf(np.zeros((N, N)), amp, M)
    assert abs(p[M // 2, M // 2] - lit / M ** 2) < 1e-15          # peak = sum A / M^2
    assert abs(p.sum() - 1.0) < 1e-12
    a = p[1:, 1:]                                                  # PSF[c+a][c+b] = PSF[c-a][c-b]
    assert np.abs(a - a[::-1, ::-1]).max() < 1e-15
    # integer tilt -> exact circular shift (t along x moves the peak to column M/2 + t)
    t = 5
    ph = np.tile(2 * np.pi * t / M * np.arange(N), (N, 1))
    q = oracle.psf(ph, amp, M)
    assert np.abs(q - np.roll(p, t, axis=1)).max() < 1e-13
    # long exposure over K identical steps = K x single
    acc = oracle.psf(ph, amp, M)
    for _ in range(2):
        oracle.psf(ph, amp, M, into=acc)
    assert np.abs(acc - 3 * q).max() < 1e-15
    # numpy cross-check with an aberrated pupil
    ph = RNG.standard_normal((N, N))
    pad = np.zeros((M, M), complex); pad[:N, :N] = amp * np.exp(1j * ph)
    ref = np.abs(np.fft.fftshift(np.fft.fft2(pad))) ** 2 / (M * M * (amp ** 2).sum())
    assert np.abs(oracle.psf(ph, amp, M) - ref).max() < 1e-14


def test_elt_psf_peak_value_golden():
    N, M, lit, peak = GOLD["psf_peak"]
    amp = inputs.annulus_mask(N, 0.04, 19.2, 5.5)
    assert int(amp.sum()) == lit and lit / M ** 2 == peak


# ----------------------------------------------------------------------------- noise
def _curand_host_philox(seed, n_words, offset=0):
    path = None
    for cand in ("/usr/local/cuda/lib64/libcurand.so", "libcurand.so", "libcurand.so.10"):
        try:
            path = C.CDLL(cand); break
        except OSError:
            continue
    if path is None:
        return None
    gen = C.c_void_p()
    if path.curandCreateGeneratorHost(C.byref(gen), 161) != 0:      # CURAND_RNG_PSEUDO_PHILOX4_32_10 = 161
        return None
    assert path.curandSetPseudoRandomGeneratorSeed(gen, C.c_ulonglong(seed)) == 0
    if offset:
        assert path.curandSetGeneratorOffset(gen, C.c_ulonglong(offset)) == 0
    out = np.empty(n_words, dtype=np.uint32)
    assert path.curandGenerate(gen, out.ctypes.data_as(C.POINTER(C.c_uint)), C.c_size_t(n_words)) == 0
    path.curandDestroyGenerator(gen)
    return out


def test_philox_matches_curand_host_generator():
    """Bit-stream pin: cuRAND's host Philox4_32_10 (a library; needs no GPU) emits, for seed s, in its
    default ordering, group g of four words = philox(counter = (g // 65536, 0, g % 65536, 0),
    key = (s lo, s hi)): 65536 interleaved subsequences (counter word 2), each advancing counter word 0."""
    seed = 0x0123456789ABCDEF
    n_groups = 65536 + 8
    ref = _curand_host_philox(seed, 4 * n_groups)
    if ref is None:
        pytest.skip("libcurand host generator not available")
    key = [seed & 0xFFFFFFFF, seed >> 32]
    for g in list(range(24)) + [4095, 65535, 65536, 65537, 65543]:
        got = oracle.philox4x32_10([g // 65536, 0, g % 65536, 0], key)
        assert np.array_equal(got, ref[4 * g:4 * g + 4]), g
    seed2 = 42
    ref2 = _curand_host_philox(seed2, 8)
    assert np.array_equal(oracle.philox4x32_10([0, 0, 1, 0], [42, 0]), ref2[4:8])
    # an offset of 2^50 words = 2^32 positions in each of the 65536 subsequences: counter word 1 = 1
    ref3 = _curand_host_philox(seed, 12, offset=(1 << 50) + 4 * 65536 * 5)
    assert np.array_equal(oracle.philox4x32_10([5, 1, 0, 0], key), ref3[0:4])
    assert np.array_equal(oracle.philox4x32_10([5, 1, 2, 0], key), ref3[8:12])


def test_philox_uses_all_counter_and_key_words():
    base = oracle.philox4x32_10([1, 2, 3, 4], [5, 6])
    for i in range(4):
        c = [1, 2, 3, 4]; c[i] += 1
        assert not np.array_equal(oracle.philox4x32_10(c, [5, 6]), base)
    assert not np.array_equal(oracle.philox4x32_10([1, 2, 3, 4], [5, 7]), base)
    assert not np.array_equal(oracle.philox4x32_10([1, 2, 3, 4], [6, 6]), base)


def test_noise_poisson_is_inverse_cdf_and_gaussian_is_box_muller():
    from scipy.stats import poisson
    P, n_img = 8, 40
    img = RNG.uniform(0.0, 0.3, (n_img, P, P))
    img[0] = 0.0
    seed, src, step, nph, ron = 991, 3, 17, 1000.0, 3.0
    noisy, counts = oracle.noise(img, None, seed, src, step, nph, ron)
    key = [seed & 0xFFFFFFFF, seed >> 32]
    mu = nph * img
    for sa in (0, 1, 7, 39):
        for px in (0, 5, 63):
            w = oracle.philox4x32_10([px, sa, src, step], key)
            u = ((w >> 8).astype(np.float64) + 0.5) / 2 ** 24
            m = mu[sa].ravel()[px]
            k_ref = int(poisson.ppf(u[0], m)) if m > 0 else 0      # library inverse CDF
            assert counts[sa].ravel()[px] == k_ref
            z = math.sqrt(-2 * math.log(u[1])) * math.cos(2 * math.pi * u[2])
            assert abs(noisy[sa].ravel()[px] - (k_ref + ron * z)) < 1e-12
    assert np.all(counts[0] == 0)
    # statistics: (noisy - mu) has mean 0 and variance mu + ron^2 (4 sigma)
    r = (noisy - mu).ravel()
    var_expected = (mu + ron ** 2).ravel()
    zscore = r.sum() / math.sqrt(var_expected.sum())
    assert abs(zscore) < 4.0
    chi = (r ** 2 / var_expected).mean()
    assert abs(chi - 1.0) < 4.0 * math.sqrt(2.5 / r.size)


def test_noise_skips_invalid_subapertures_and_full_cdf_range():
    img = np.full((2, 4, 4), 0.05)
    valid = np.array([1, 0], dtype=np.uint8)
    noisy, counts = oracle.noise(img, valid, 5, 0, 0, 1000.0, 3.0)
    assert np.all(noisy[1] == 0.0) and np.all(counts[1] == 0) and counts[0].mean() > 20
    # bright pixel (mu = 300: exp(-mu) underflows fp32 but not fp64)
    noisy, counts = oracle.noise(np.full((1, 8, 8), 0.3), None, 5, 0, 0, 1000.0, 0.0)
    assert abs(counts.mean() - 300.0) < 4 * math.sqrt(300.0 / 64)


@pytest.mark.parametrize("mu", [63.9, 64.0, 100.5, 226.7, 744.0, 746.0, 800.0, 1026.3, 1e4])
def test_poisson_inverse_cdf_matches_scipy_for_bright_pixels(mu):
    """Reading O5 (revised): the Poisson draw is the inverse CDF at u for EVERY mean.  exp(-mu) underflows FP64 above
    mu ~ 745, where a search from k = 0 returns floor(mu)+1 for every u; the oracle searches from the mode instead.
    Library routine: scipy.stats.poisson.ppf; statistics: mean and variance of the counts equal mu."""
    from scipy.stats import poisson
    P, n_img, seed, src, step = 16, 40, 77, 2, 5
    img = np.full((n_img, P, P), 1.0)
    _, counts = oracle.noise(img, None, seed, src, step, mu, 0.0)              # photons = mu, image = 1
    key = [seed & 0xFFFFFFFF, seed >> 32]
    for sa in (0, 3, 39):
        for px in range(0, P * P, 5):
            w = oracle.philox4x32_10([px, sa, src, step], key)
            u = ((int(w[0]) >> 8) + 0.5) / 2 ** 24
            assert counts[sa].ravel()[px] == int(poisson.ppf(u, mu)), (mu, u)
    c = counts.astype(np.float64).ravel()
    n = c.size
    assert abs(c.mean() - mu) < 4.0 * math.sqrt(mu / n)
    assert abs(c.var() / mu - 1.0) < 4.0 * math.sqrt(2.0 / n) + 1.0 / mu          # a constant floor(mu)+1 would give 0


def test_poisson_inverse_cdf_tails():
    """Extreme u (the ends of the 24-bit lattice) at small and large means, through the exported entry point: a
    one-pixel image and a search over Philox counters for the smallest and largest u of a few thousand draws."""
    from scipy.stats import poisson
    for mu in (3.0, 90.0, 2000.0):
        img = np.full((200, 4, 4), 1.0)
        _, counts = oracle.noise(img, None, 11, 0, 0, mu, 0.0)
        key = [11, 0]
        us = np.array([[((int(oracle.philox4x32_10([px, sa, 0, 0], key)[0]) >> 8) + 0.5) / 2 ** 24
                        for px in range(16)] for sa in range(200)])
        for idx in (np.unravel_index(us.argmin(), us.shape), np.unravel_index(us.argmax(), us.shape)):
            assert counts[idx[0]].ravel()[idx[1]] == int(poisson.ppf(us[idx], mu)), (mu, us[idx])


# ----------------------------------------------------------------------------- input generator (harness)
def test_screen_generator_variance_and_structure_function():
    n, d = 256, 0.1
    exp_var = inputs.screen_expected_variance(n, d, inputs.R0_REF, inputs.L0_REF)
    # continuous-spectrum value 0.08633 (L0/r0)^(5/3) is an upper bound the discrete sum approaches
    cont = 0.0229 * 2 * math.pi * (3.0 / 5.0) * (inputs.L0_REF / inputs.R0_REF) ** (5.0 / 3.0)
    assert 0.5 * cont < exp_var < cont
    rng = np.random.default_rng(3)
    var, sf = [], []
    for _ in range(6):
        a, b = inputs.von_karman_pair(n, d, inputs.R0_REF, inputs.L0_REF, rng)
        for s in (a, b):
            s = s.astype(np.float64)
            var.append(s.var())
            sf.append(((s[:, 3:] - s[:, :-3]) ** 2).mean())
    assert abs(np.mean(var) / exp_var - 1.0) < 0.15
    # D(rho) -> 6.88 (rho/r0)^(5/3) for d << rho << L0 (outer scale lowers it somewhat)
    kolm = 6.88 * (3 * d / inputs.R0_REF) ** (5.0 / 3.0)
    assert 0.6 * kolm < np.mean(sf) < 1.05 * kolm


def test_configs_have_survey_shapes():
    c2 = inputs.make_config(2, with_screens=False)
    assert c2.pupil.n == 960 and c2.wfs[0].n_grid == 1280 and len(c2.layers) == 10
    assert abs(c2.grid_pitch(0) - 0.03) < 1e-15 and len(c2.sources) == 6
    c3 = inputs.make_config(3, with_screens=False)
    assert c3.wfs[1].fft == 1024 and c3.wfs[1].n_samp == 480 and c3.wfs[1].n_pix == 128
    assert c3.psf_fft == 2048 and len(c3.science_sources()) == 10 and len(c3.sources) == 19
    c4 = inputs.make_config(4, with_screens=False, lgs_fft=64)
    assert len(c4.layers) == 35 and c4.layers[0].n == 8192 and c4.wfs[0].n_samp == 32
    assert abs(sum(l.weight for l in c4.layers) - 1.0) < 1e-12 and len(c4.sources) == 10
    c1 = inputs.make_config(1, with_screens=False)
    assert c1.wfs[0].fft == 24 and c1.pupil.r_in_m == 5.5 and c1.pupil.r_out_m == 19.2


# ----------------------------------------------------------------------------- phase maps
@pytest.mark.parametrize("entry", [e for e in GOLD["cog"] if e[0] == (8, 16, 2, 8)])
def test_phase_map_tilt_on_flat_atmosphere_gives_golden_cog(entry):
    """A static map alpha * j summed to the (flat) open-loop wavefront is a pure x-tilt of alpha rad/sample: every
    fully lit subaperture of c0 must show the closed-form CoG of SURVEY.md section 8(c), and no y-slope."""
    (n, M, beta, P), t, cog = entry
    cfg = inputs.make_config(0)
    cfg.layers[0].screen = np.zeros_like(cfg.layers[0].screen)
    N = cfg.wfs[0].n_sub * n
    alpha = 2.0 * np.pi * t / M
    cfg.phase_maps = {0: np.tile((alpha * np.arange(N)).astype(np.float64), (N, 1))}
    res = oracle.forward(cfg, 0, 1)
    assert np.allclose(res["phase"][0][0], cfg.phase_maps[0], atol=0.0)
    amp = cfg.wfs[0].amp.reshape(cfg.wfs[0].n_sub, n, cfg.wfs[0].n_sub, n)
    full = (amp.min(axis=(1, 3)) == 1.0).ravel()
    assert full.sum() == 60                                   # 60 fully lit subapertures
    sx, sy = res["slopes"][0][0]
    assert np.abs(sx[full] - cog).max() < 1e-10 and np.abs(sy[full]).max() < 1e-10


def test_phase_map_adds_to_phase_and_piston_map_changes_nothing_else():
    cfg = inputs.make_config(0)
    base = oracle.forward(cfg, 3, 1)
    rng = np.random.default_rng(5)
    N = cfg.grid_n(0)
    m = rng.normal(size=(N, N)).astype(np.float32)
    cfg.phase_maps = {0: m}
    with_map = oracle.forward(cfg, 3, 1)
    assert np.array_equal(with_map["phase"][0][0], base["phase"][0][0] + m.astype(np.float64))
    assert np.abs(with_map["slopes"][0] - base["slopes"][0]).max() > 1e-3          # a random map does move the spots
    cfg.phase_maps = {0: np.full((N, N), 1.2345, np.float32)}                       # piston: invisible to |FFT|^2
    piston = oracle.forward(cfg, 3, 1)
    assert np.abs(piston["images"][0] - base["images"][0]).max() < 1e-12
    assert np.abs(piston["slopes"][0] - base["slopes"][0]).max() < 1e-10


# ----------------------------------------------------------------------------- residual-phase entry
def test_modes_to_map_brute_force_one_hot_and_linearity():
    rng = np.random.default_rng(8)
    modes = rng.normal(size=(5, 7, 3))
    c = rng.normal(size=5)
    got = oracle.modes_to_map(modes, c, -1.0)
    want = np.zeros((7, 3))
    for m in range(5):                                     # brute force, the definition written out
        for i in range(7):
            for j in range(3):
                want[i, j] -= c[m] * modes[m, i, j]
    assert np.abs(got - want).max() < 1e-14
    one_hot = np.zeros(5); one_hot[3] = 2.5
    assert np.array_equal(oracle.modes_to_map(modes, one_hot, 1.0), 2.5 * modes[3])
    c2 = rng.normal(size=5)
    assert np.abs(oracle.modes_to_map(modes, c + c2, 1.0) - oracle.modes_to_map(modes, c, 1.0)
                  - oracle.modes_to_map(modes, c2, 1.0)).max() < 1e-14


def test_residual_of_a_tilt_mode_cancels_a_tilted_wavefront():
    """Closed loop in one line: open-loop tilt from a linear screen, minus coefficient x tilt mode with
    the matching coefficient, leaves a flat residual: zero slopes on every valid subaperture."""
    cfg = inputs.make_config(0)
    g_px = 0.125
    cfg.layers[0].screen = inputs.linear_screen(cfg.layers[0].n, 0.0, 0.0, g_px)
    N = cfg.grid_n(0)
    alpha = g_px * cfg.grid_pitch(0) / cfg.layers[0].pitch_m * cfg.lambda_ref_m / cfg.sources[0].lambda_m
    mode = np.tile(np.arange(N, dtype=np.float64), (N, 1))[None]          # unit x-ramp, radians per sample
    open_loop = oracle.forward(cfg, 0, 1)
    assert np.abs(open_loop["slopes"][0][0][0]).max() > 0.05
    cfg.phase_maps = {0: oracle.modes_to_map(mode, np.array([alpha]), -1.0)}
    closed = oracle.forward(cfg, 0, 1)
    assert np.abs(closed["slopes"][0]).max() < 1e-9


# ----------------------------------------------------------------------------- Strehl on the PSF
def test_strehl_flat_is_one_tilt_is_zero_and_marechal_for_small_aberrations():
    N, M = 48, 128
    amp = inputs.annulus_mask(N, 0.1, 2.4, 0.7)
    flat = oracle.psf(np.zeros((N, N)), amp, M)
    assert abs(oracle.strehl(flat, amp, 1) - 1.0) < 1e-12                       # diffraction limit
    assert abs(oracle.strehl(3.0 * flat, amp, 3) - 1.0) < 1e-12                 # long exposure of 3 equal steps
    tilt = np.tile(2.0 * np.pi * 8 * np.arange(N) / M, (N, 1))                  # spot moved 8 pixels away: peak pixel ~ empty
    assert oracle.strehl(oracle.psf(tilt, amp, M), amp, 1) < 1e-3
    rng = np.random.default_rng(4)
    for sigma in (0.05, 0.1, 0.2):                                              # Marechal: S = exp(-sigma^2) + O(sigma^4 / N_lit)
        ph = rng.normal(scale=sigma, size=(N, N))
        lit = amp > 0
        var = ph[lit].var()
        s = oracle.strehl(oracle.psf(ph, amp, M), amp, 1)
        assert abs(s - np.exp(-var)) < 0.02 * var + 1e-4, (sigma, s, np.exp(-var))


def test_marechal_strehl_closed_forms_and_agreement_with_the_psf_strehl():
    N, M = 48, 128
    amp = inputs.annulus_mask(N, 0.1, 2.4, 0.7)
    assert oracle.strehl_marechal(np.full((N, N), 7.5), amp) == 1.0             # piston only
    two = np.where(np.arange(N)[None, :] < N // 2, -0.3, 0.3) * np.ones((N, 1))  # two-level phase +-a on a symmetric pupil
    assert abs(oracle.strehl_marechal(two, amp) - np.exp(-0.09)) < 1e-12          # variance a^2
    # outside the pupil the phase does not count
    junk = two + 100.0 * (amp == 0)
    assert abs(oracle.strehl_marechal(junk, amp) - np.exp(-0.09)) < 1e-12
    rng = np.random.default_rng(6)
    ph = rng.normal(scale=0.15, size=(N, N))
    s_psf = oracle.strehl(oracle.psf(ph, amp, M), amp, 1)
    assert abs(oracle.strehl_marechal(ph, amp) - s_psf) < 2e-3                    # the two estimates of PAPER.md:86 agree


# ----------------------------------------------------------------------------- step driver wiring (O2 t_k, O5 counter)
def test_forward_time_and_noise_counter_use_the_absolute_step_index():
    """oracle.forward(step0 = 7, n_steps = 2): entry k = 1 is time t = (7 + 1) dt and its
    noise counter is (pixel, subaperture, GLOBAL source index, 7 + 1) (O5).  Compared with direct calls of the pinned
    pieces, on a workload whose wind moves the footprint by a non-integer number of pixels per step and whose sensor
    sources are not source 0, so that t = k dt, a local source index or step k instead of step0 + k all fail."""
    cfg = inputs.make_config(2, n_sub=6, screen_n=128, n_steps=2, n_layers=3)
    cfg.sources = cfg.sources[3:5]                       # global indices 0, 1 of this config; keep two LGS
    cfg.noise = inputs.Noise(seed=0x1234567890ABCDEF, photons_per_subap=1000.0, read_noise_e=3.0)
    res = oracle.forward(cfg, 7, 2, noise_on=True)
    W = cfg.wfs[0]
    for s in (0, 1):
        src = cfg.sources[s]
        for k in (0, 1):
            t = (7 + k) * cfg.dt_s
            ph = oracle.trace(cfg.layers, src.theta_x_rad, src.theta_y_rad, src.altitude_m, src.lambda_m,
                              cfg.lambda_ref_m, cfg.grid_n(s), cfg.grid_pitch(s), t)
            assert np.array_equal(res["phase"][s][k], ph)
            wrong = oracle.trace(cfg.layers, src.theta_x_rad, src.theta_y_rad, src.altitude_m, src.lambda_m,
                                 cfg.lambda_ref_m, cfg.grid_n(s), cfg.grid_pitch(s), k * cfg.dt_s)
            assert np.abs(wrong - ph).max() > 1e-3       # the pin can tell t = k dt from t = (step0 + k) dt
            img, valid = oracle.sh_images(ph, W.amp, W.n_sub, W.n_samp, W.fft, W.bin, W.n_pix, W.min_illum)
            assert np.array_equal(res["images"][s][k], img)
            nz, ct = oracle.noise(img, valid, cfg.noise.seed, s, 7 + k, 1000.0, 3.0)
            assert np.array_equal(res["counts"][s][k], ct) and np.array_equal(res["noisy"][s][k], nz)
            for bad_src, bad_step in ((s, k), (1 - s, 7 + k), (s, 7)):
                if (bad_src, bad_step) != (s, 7 + k):
                    assert not np.array_equal(oracle.noise(img, valid, cfg.noise.seed, bad_src, bad_step, 1000.0, 3.0)[1], ct)
            assert np.array_equal(res["slopes"][s][k], oracle.centroids(nz, valid))
    only1 = oracle.forward(cfg, 7, 2, noise_on=True, sources=[1])      # a subset keeps the global source index
    assert list(only1["counts"].keys()) == [1] and np.array_equal(only1["counts"][1], res["counts"][1])


# ----------------------------------------------------------------------------- SH image on the M > 64 branch (O3, O4)
def test_big_fft_sensor_image_closed_form_flat_and_integer_tilt():
    """aoref_sh_images takes its radix-2 branch for M > 64 (the NGS sensors).  Flat n = 48, M = 128, beta = 8, P = 16:
    the image is the outer product of the binned Dirichlet profile (normalisation 1/(M^2 n^2), full window, bin 8);
    an x-tilt of exactly one detector pixel (alpha = 2 pi beta / M) shifts the whole image one column to the right,
    and a cropped window (P = 8: the central 64 of 128 FFT pixels) is the centre of the full image."""
    n, M, beta, P = 48, 128, 8, 16
    prof = dirichlet_binned(n, M, beta, P, 0.0)
    img, valid = one_subap(np.zeros((n, n)), n, M, beta, P)
    assert valid == 1 and abs(prof.sum() - 1.0) < 1e-12
    assert np.abs(img - np.outer(prof, prof)).max() < 1e-13
    a = 2.0 * np.pi * beta / M
    tilt = np.tile(a * np.arange(n), (n, 1))                        # phase = alpha * column index
    img_t, _ = one_subap(tilt, n, M, beta, P)
    px = dirichlet_binned(n, M, beta, P, a)
    assert np.abs(img_t - np.outer(prof, px)).max() < 1e-13        # rows unchanged, columns carry the tilt
    assert np.abs(px - np.roll(prof, 1)).max() < 1e-13              # integer shift of the periodic image
    half, _ = one_subap(np.zeros((n, n)), n, M, beta, 8)
    assert np.abs(half - img[4:12, 4:12]).max() < 1e-14
    # y-tilt goes to the rows (orientation), two subapertures side by side are independent
    ph2 = np.zeros((2 * n, 2 * n)); ph2[:n, n:] = tilt.T
    img2, v2 = oracle.sh_images(ph2, np.ones((2 * n, 2 * n), np.float32), 2, n, M, beta, P, 0.0)
    assert np.abs(img2[1] - np.outer(px, prof)).max() < 1e-13 and np.abs(img2[0] - np.outer(prof, prof)).max() < 1e-13


# ----------------------------------------------------------------------------- NEXT-4: polychromatic PSF (reading O8)
def _dirichlet_scaled(N, M, s):
    """|sum_{a<N} exp(-2 pi i s kappa a / M)|^2 = sin^2(N psi/2)/sin^2(psi/2), psi = 2 pi s kappa/M, kappa = k - M/2."""
    psi = 2.0 * np.pi * s * (np.arange(M) - M / 2.0) / M
    sn = np.sin(psi / 2.0)
    with np.errstate(all="ignore"):
        return np.where(np.abs(sn) < 1e-13, float(N * N), np.sin(N * psi / 2.0) ** 2 / sn ** 2)


def test_psf_poly_one_wavelength_is_the_monochromatic_psf():
    N, M = 24, 64
    amp = inputs.annulus_mask(N, 0.04, N * 0.02, 0.12)
    ph = RNG.standard_normal((N, N))
    mono = oracle.psf(ph, amp, M)
    poly = oracle.psf_poly(ph, amp, M, 2.2e-6, [2.2e-6], [1.0])
    assert np.abs(poly - mono).max() < 1e-13
    acc = oracle.psf_poly(ph, amp, M, 2.2e-6, [2.2e-6], [0.25], into=mono.copy())       # accumulates, weights scale
    assert np.abs(acc - 1.25 * mono).max() < 1e-13


def test_psf_poly_flat_square_pupil_is_the_weighted_sum_of_scaled_dirichlet_products():
    """Two wavelengths on a flat square pupil: each contributes w_j s_j^2 D(s_j kappa_k) D(s_j kappa_m) / (M^2 N^2), a
    diffraction pattern 1/s_j times wider on the fixed pixel grid (the lambda-dependent pixel scale), peak w_j s_j^2 N^2/M^2."""
    N, M, lam_s = 10, 48, 2.0e-6
    lams, wts = [1.6e-6, 2.5e-6], [0.7, 0.3]
    p = oracle.psf_poly(np.zeros((N, N)), np.ones((N, N), np.float32), M, lam_s, lams, wts)
    want = np.zeros((M, M))
    for lam, w in zip(lams, wts):
        s = lam_s / lam
        D = _dirichlet_scaled(N, M, s)
        want += w * s * s * np.outer(D, D) / (M * M * N * N)
    assert np.abs(p - want).max() < 1e-13
    assert abs(p[M // 2, M // 2] - sum(w * (lam_s / l) ** 2 for l, w in zip(lams, wts)) * N * N / M ** 2) < 1e-14
    # first zero of the longer wavelength is further out: kappa = M / (N s)
    s_long = lam_s / 2.5e-6
    only = oracle.psf_poly(np.zeros((N, N)), np.ones((N, N), np.float32), M, lam_s, [2.5e-6], [1.0])
    assert abs(M / (N * s_long) - 6.0) < 1e-12 and only[M // 2, M // 2 + 6] < 1e-28 < only[M // 2, M // 2 + 5]


def test_psf_poly_twice_the_wavelength_is_the_central_crop_of_the_2M_transform():
    """s = 1/2: exp(-2 pi i kappa a / (2M)) is the pixel-centred DFT of size 2M, so the PSF at lambda = 2 lambda_s on
    M pixels equals the central M x M crop of aoref_psf at size 2M of the phase scaled by 1/2 (normalisation included:
    s^2 / M^2 = 1 / (2M)^2).  An independent route through the pinned C transform."""
    N, M = 20, 32
    amp = inputs.annulus_mask(N, 0.04, N * 0.02, 0.1)
    ph = RNG.standard_normal((N, N)) * 2.0
    poly = oracle.psf_poly(ph, amp, M, 1.0e-6, [2.0e-6], [1.0])
    big = oracle.psf(0.5 * ph, amp, 2 * M)
    assert np.abs(poly - big[M // 2:M // 2 + M, M // 2:M // 2 + M]).max() < 1e-13


def test_psf_poly_tilt_is_achromatic_in_angle_and_energy_stays_in_the_field():
    """A tilt of optical path moves every wavelength to the same detector pixel (phase scales with s, so does the
    frequency axis); and a compact PSF keeps sum = sum of weights to the part that leaves the field."""
    N, M, lam_s = 16, 64, 1.0e-6
    t = 7
    ph = np.tile(2 * np.pi * t / M * np.arange(N), (N, 1))                     # radians at lambda_s
    for lam in (0.8e-6, 1.0e-6, 1.7e-6):
        p = oracle.psf_poly(ph, np.ones((N, N), np.float32), M, lam_s, [lam], [1.0])
        assert np.unravel_index(np.argmax(p), p.shape) == (M // 2, M // 2 + t)
    ph = RNG.standard_normal((N, N)) * 0.3
    p = oracle.psf_poly(ph, np.ones((N, N), np.float32), 8 * N, lam_s, [1.5e-6, 2.0e-6], [0.6, 0.4])
    assert 0.93 < p.sum() <= 1.0 + 1e-12                                        # wider than one period never happens for s < 1
    res = oracle.forward(_poly_cfg(), 0, 2, want_wfs=False)
    assert set(res["psf"]) == {0}


def _poly_cfg():
    cfg = inputs.make_config(3, n_sub=4, screen_n=128, n_steps=2, n_layers=2)
    cfg.sources = [cfg.sources[-1]]; cfg.sources[0].wfs_index = -1
    cfg.wfs = []
    cfg.psf_band = ([2.0e-6, 2.2e-6, 2.4e-6], [0.3, 0.4, 0.3])
    return cfg


def test_forward_uses_the_band_for_every_step_of_the_long_exposure():
    cfg = _poly_cfg()
    res = oracle.forward(cfg, 3, 2, want_wfs=False)
    want = np.zeros((cfg.psf_fft, cfg.psf_fft))
    for k in range(2):
        oracle.psf_poly(res["phase"][0][k], cfg.pupil.amp, cfg.psf_fft, cfg.sources[0].lambda_m, *cfg.psf_band, into=want)
    assert np.array_equal(res["psf"][0], want)
    cfg.psf_band = None
    mono = oracle.forward(cfg, 3, 2, want_wfs=False)["psf"][0]
    assert np.abs(mono - want).max() > 1e-6                                     # the band does change the image


# ----------------------------------------------------------------------------- NEXT-3: LGS elongation (reading O9)
def _elong(phase, n_sub, n, M, beta, P, z, rho, launch=(0.0, 0.0), d=0.03, lam=589e-9, H=90e3, amp=None):
    amp = np.ones((n_sub * n, n_sub * n), np.float32) if amp is None else amp
    return oracle.sh_images_elong(phase, amp, n_sub, n, M, beta, P, 0.5, d, lam, H, launch, z, rho)


def test_elongation_delta_profile_at_the_focus_altitude_changes_nothing():
    n_sub, n, M, beta, P = 4, 8, 16, 2, 8
    ph = RNG.standard_normal((n_sub * n, n_sub * n))
    amp = inputs.annulus_mask(n_sub * n, 0.03, n_sub * n * 0.015, 0.1)
    ref, v0 = oracle.sh_images(ph, amp, n_sub, n, M, beta, P, 0.5)
    img, v1 = _elong(ph, n_sub, n, M, beta, P, [90e3], [1.0], launch=(3.0, -2.0), amp=amp)
    assert np.array_equal(v0, v1) and np.array_equal(img, ref)
    # several scatterers, all at H: still the point-beacon image (weights sum to 1)
    img2, _ = _elong(ph, n_sub, n, M, beta, P, [90e3] * 3, [0.2, 0.5, 0.3], launch=(3.0, -2.0), amp=amp)
    assert np.abs(img2 - ref).max() < 1e-15


def test_elongation_is_a_whole_pixel_shift_along_the_launch_to_subaperture_direction():
    """One scatterer above the focus altitude, chosen so that the spot of the subaperture one pitch to the right of the
    launch point moves by exactly one detector pixel: delta = (c - L)(1/H - 1/z), shift = delta M d / lambda FFT pixels.
    The shift grows linearly with the baseline, points away from the launch point for z > H (towards it for z < H), and
    is along y for subapertures above / below the launch point."""
    n_sub, n, M, beta, P, d, lam, H = 5, 8, 16, 2, 8, 0.05, 589e-9, 90e3
    N = n_sub * n
    ph = np.zeros((N, N))
    base, _ = oracle.sh_images(ph, np.ones((N, N), np.float32), n_sub, n, M, beta, P, 0.5)
    pitch = n * d                                                  # distance between subaperture centres
    # launch at the centre of subaperture (2, 2) = the grid centre; one-pixel shift (beta FFT pixels) per pitch
    inv = 1.0 / H - beta * lam / (M * d * pitch)                   # 1/z with (1/H - 1/z) pitch M d / lambda = beta
    z = 1.0 / inv
    assert z > H
    img, _ = _elong(ph, n_sub, n, M, beta, P, [z], [1.0], d=d, lam=lam, H=H)
    sub = lambda p, q: img[p * n_sub + q]
    assert np.abs(sub(2, 2) - base[0]).max() < 1e-14                                   # on the launch axis: no shift
    assert np.abs(sub(2, 3) - np.roll(base[0], 1, axis=1)).max() < 1e-13               # +x neighbour: one pixel to +x
    assert np.abs(sub(2, 4) - np.roll(base[0], 2, axis=1)).max() < 1e-13               # twice the baseline: two pixels
    assert np.abs(sub(2, 1) - np.roll(base[0], -1, axis=1)).max() < 1e-13              # -x neighbour: to -x
    assert np.abs(sub(3, 2) - np.roll(base[0], 1, axis=0)).max() < 1e-13               # +y neighbour: rows
    assert np.abs(sub(0, 4) - np.roll(np.roll(base[0], -2, axis=0), 2, axis=1)).max() < 1e-13
    # below the focus altitude the spot moves towards the launch point
    z_lo = 1.0 / (1.0 / H + beta * lam / (M * d * pitch))
    lo, _ = _elong(ph, n_sub, n, M, beta, P, [z_lo], [1.0], d=d, lam=lam, H=H)
    assert np.abs(lo[2 * n_sub + 3] - np.roll(base[0], -1, axis=1)).max() < 1e-13
    # a launch point moved by one pitch moves the pattern with it
    off, _ = _elong(ph, n_sub, n, M, beta, P, [z], [1.0], launch=(pitch, 0.0), d=d, lam=lam, H=H)
    assert np.abs(off[2 * n_sub + 3] - base[0]).max() < 1e-13 and np.abs(off[2 * n_sub + 2] - np.roll(base[0], -1, axis=1)).max() < 1e-13


def test_elongated_image_is_the_profile_weighted_sum_and_conserves_energy():
    n_sub, n, M, beta, P, d, lam, H = 5, 8, 16, 2, 8, 0.05, 589e-9, 90e3
    N = n_sub * n
    ph = RNG.standard_normal((N, N)) * 0.7
    amp = inputs.annulus_mask(N, d, N * d / 2, 0.3)
    z = np.array([84e3, 88e3, 90e3, 93e3, 97e3]); rho = np.array([0.1, 0.25, 0.3, 0.2, 0.15])
    img, valid = _elong(ph, n_sub, n, M, beta, P, z, rho, launch=(-0.4, 0.9), d=d, lam=lam, H=H, amp=amp)
    parts = [_elong(ph, n_sub, n, M, beta, P, [zi], [1.0], launch=(-0.4, 0.9), d=d, lam=lam, H=H, amp=amp)[0] for zi in z]
    assert np.abs(img - sum(r * p for r, p in zip(rho, parts))).max() < 1e-15         # incoherent sum over the column
    point, _ = oracle.sh_images(ph, amp, n_sub, n, M, beta, P, 0.5)
    assert np.abs(img.sum(axis=(1, 2)) - point.sum(axis=(1, 2))).max() < 1e-13         # full window: Parseval per scatterer
    # the spot is longer along the baseline: second moment along c - L grows, across it it does not shrink the energy
    far = 0 * n_sub + 4 if valid[4] else int(np.flatnonzero(valid)[0])
    assert img[far].max() < point[far].max()


def test_forward_picks_the_profile_of_the_absolute_step():
    cfg = inputs.make_config(2, n_sub=6, screen_n=128, n_steps=2, n_layers=2)
    cfg.sources = cfg.sources[:2]
    cfg.sodium = inputs.sodium_profile(cfg, n_z=3, n_t=4, launch="side")
    assert cfg.sodium.rho.shape == (4, 3) and np.allclose(cfg.sodium.rho.sum(axis=1), 1.0)
    res = oracle.forward(cfg, 6, 2)
    W = cfg.wfs[0]
    for s in (0, 1):
        for k in (0, 1):
            img, _ = oracle.sh_images_elong(res["phase"][s][k], W.amp, W.n_sub, W.n_samp, W.fft, W.bin, W.n_pix, W.min_illum,
                                            cfg.grid_pitch(s), cfg.sources[s].lambda_m, cfg.sources[s].altitude_m,
                                            cfg.sodium.launch_xy_m[s], cfg.sodium.z_m, cfg.sodium.rho[(6 + k) % 4])
            assert np.array_equal(res["images"][s][k], img)
            other, _ = oracle.sh_images_elong(res["phase"][s][k], W.amp, W.n_sub, W.n_samp, W.fft, W.bin, W.n_pix, W.min_illum,
                                              cfg.grid_pitch(s), cfg.sources[s].lambda_m, cfg.sources[s].altitude_m,
                                              cfg.sodium.launch_xy_m[s], cfg.sodium.z_m, cfg.sodium.rho[k % 4])
            assert not np.array_equal(other, img)
