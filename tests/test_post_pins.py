"""Pins for oracle/post_oracle.py (multi-template median combination; Monte-Carlo
limiting flux) against things other than itself.  CPU only."""
import math
import statistics

import numpy as np
import pytest

from oracle import post_oracle as po


@pytest.mark.parametrize("n", [1, 2, 3, 4, 5, 7, 8])
def test_median_matches_statistics_median_on_small_stacks(n):
    rng = np.random.default_rng(n)
    Ds = [rng.standard_normal((5, 7)) for _ in range(n)]
    sc = rng.uniform(0.5, 2.0, n)
    out = po.median_combine(Ds, sc)
    for y in range(5):
        for x in range(7):
            assert out[y, x] == pytest.approx(statistics.median([sc[k] * Ds[k][y, x] for k in range(n)]), abs=0, rel=1e-15)


def test_median_known_values_and_invariances():
    # order statistics of a hand-written stack
    vals = [[3.0, -1.0], [1.0, 5.0], [2.0, 0.0], [10.0, 4.0], [-7.0, 2.0]]
    Ds = [np.array([v]) for v in vals]
    out = po.median_combine(Ds, [1.0] * 5)
    assert out.tolist() == [[2.0, 2.0]]
    # permutation invariance, positive scaling commutes with the median
    perm = [4, 2, 0, 3, 1]
    assert np.array_equal(po.median_combine([Ds[i] for i in perm], [1.0] * 5), out)
    assert np.array_equal(po.median_combine(Ds, [3.0] * 5), 3.0 * out)
    # the scale belongs to the image it multiplies
    out2 = po.median_combine(Ds, [1.0, 1.0, 1.0, 0.1, 1.0])   # 10 -> 1, 4 -> 0.4
    assert out2.tolist() == [[1.0, 0.4]]


def test_median_nan_reading_M2_matches_numpy_median():
    """A NaN in any image makes the pixel NaN -- numpy.median's behaviour (library routine)."""
    rng = np.random.default_rng(4)
    for n in (3, 4, 5):
        Ds = [rng.standard_normal((6, 7)) for _ in range(n)]
        Ds[1][2, 3] = np.nan
        Ds[n - 1][0, 0] = np.nan
        Ds[0][0, 0] = np.nan
        out = po.median_combine(Ds, [1.0] * n)
        ref = np.median(np.stack(Ds), axis=0)
        assert np.isnan(out[2, 3]) and np.isnan(out[0, 0]) and np.isnan(out).sum() == 2
        assert np.array_equal(out, ref, equal_nan=True)


@pytest.mark.parametrize("r,count", [(1.0, 5), (2.0, 13), (3.0, 29), (4.0, 49), (5.0, 81), (1.5, 9), (2.5, 21)])
def test_disc_pixel_count_is_the_gauss_circle_number(r, count):
    """N(r) = #{(i,j) in Z^2 : i^2 + j^2 <= r^2}: 5, 13, 29, 49, 81 for r = 1..5 (OEIS A000328)."""
    D = np.ones((41, 41))
    assert po.aperture_flux(D, None, 20.0, 20.0, r) == count
    assert po.aperture_flux(7.5 * D, None, 20.0, 20.0, r) == 7.5 * count


def test_linear_ramp_flux_is_count_times_centre_value():
    y, x = np.mgrid[0:40, 0:50].astype(np.float64)
    D = 3.0 + 0.25 * x - 0.5 * y
    for (x0, y0, r) in [(25, 20, 3.0), (10, 30, 5.0), (7, 7, 2.5)]:
        n = po.aperture_flux(np.ones_like(D), None, x0, y0, r)
        assert po.aperture_flux(D, None, x0, y0, r) == pytest.approx(n * D[y0, x0], rel=1e-13)
    # an off-centre position still sums exactly the pixels inside its own disc
    f = po.aperture_flux(D, None, 25.3, 19.6, 3.0)
    brute = sum(D[j, i] for j in range(40) for i in range(50) if (i - 25.3) ** 2 + (j - 19.6) ** 2 <= 9.0)
    assert f == pytest.approx(brute, rel=1e-14)


def test_frame_edge_and_mask_drop_the_position():
    D = np.ones((30, 30))
    assert math.isnan(po.aperture_flux(D, None, 2.0, 15.0, 3.0))       # leaves the frame on the left
    assert math.isnan(po.aperture_flux(D, None, 15.0, 27.5, 3.0))      # leaves it at the bottom
    assert po.aperture_flux(D, None, 3.0, 3.0, 3.0) == 29               # just inside
    mask = np.zeros((30, 30), dtype=np.uint8)
    mask[15, 17] = 1
    assert math.isnan(po.aperture_flux(D, mask, 15.0, 15.0, 3.0))      # (17,15) is inside the disc
    assert po.aperture_flux(D, mask, 15.0, 15.0, 1.5) == 9              # and outside the smaller one
    for bad in (float("nan"), float("inf"), -float("inf")):              # not a position at all: dropped
        assert math.isnan(po.aperture_flux(D, None, bad, 15.0, 3.0))
        assert math.isnan(po.aperture_flux(D, None, 15.0, bad, 3.0))


def test_stats_constant_and_white_noise():
    rng = np.random.default_rng(3)
    xs, ys = rng.uniform(10, 190, 1024), rng.uniform(10, 190, 1024)
    # constant image: every flux is 2 x (its own pixel count); at integer centres all counts are
    # N(4.2) = 57, so the scatter vanishes
    D = np.full((200, 200), 2.0)
    flux = po.aperture_stats(D, None, xs, ys, 4.2)[0]
    ones = po.aperture_stats(np.ones_like(D), None, xs, ys, 4.2)[0]
    assert np.allclose(flux, 2.0 * ones, rtol=0, atol=1e-12)
    xs_i, ys_i = np.round(xs), np.round(ys)
    _, (n, mean, sigma) = po.aperture_stats(D, None, xs_i, ys_i, 4.2)
    assert n == 1024 and mean == pytest.approx(2.0 * 57) and sigma < 1e-12
    # white noise of sigma_pix: sigma(flux) ~ sigma_pix sqrt(N) within sampling error
    noise = 5.0 * rng.standard_normal((200, 200))
    _, (n2, m2, s2) = po.aperture_stats(noise, None, xs_i, ys_i, 4.2)
    assert n2 == 1024
    assert s2 == pytest.approx(5.0 * math.sqrt(57), rel=0.12)
    # hand values (reading L5): 2.5 log10(5) = 1.7474250108..., and a 100x larger sigma is
    # exactly 5 magnitudes brighter
    assert po.limiting_magnitude(1.0, 25.0) == pytest.approx(23.2525749891600, abs=1e-12)
    assert po.limiting_magnitude(0.2, 25.0) == pytest.approx(25.0, abs=1e-12)
    assert po.limiting_magnitude(100.0, 25.0) == pytest.approx(18.2525749891600, abs=1e-12)


# --------------------------------------------------------------------------- resampling pins
IDENT = [0.0, 1.0, 0.0, 0.0, 0.0, 1.0]


def test_resample_identity_and_integer_shift_are_exact():
    rng = np.random.default_rng(8)
    img = rng.standard_normal((24, 30))
    out, outside = po.resample_affine(img, IDENT, 24, 30, a=3)
    inner = outside == 0
    assert inner[2:21, 2:27].all() and not inner[0].any() and not inner[:, -1].any()   # taps need a-1 / a pixels of margin
    assert np.array_equal(out[inner], img[inner])            # L(0) = 1, L(k) = 0: exact
    M = [4.0, 1.0, 0.0, -3.0, 0.0, 1.0]                      # x_in = x_out + 4, y_in = y_out - 3
    out, outside = po.resample_affine(img, M, 24, 30, a=3)
    for yo, xo in [(10, 10), (8, 3), (20, 20)]:
        assert outside[yo, xo] == 0 and out[yo, xo] == img[yo - 3, xo + 4]
    assert outside[0, 0] == 1 and out[0, 0] == 0.0           # y_in = -3 leaves the frame


@pytest.mark.parametrize("a", [2, 3, 4])
def test_resample_constant_and_lanczos_kernel_values(a):
    M = [0.37, 1.01, 0.02, -0.21, -0.015, 0.99]
    out, outside = po.resample_affine(np.full((40, 40), 7.25), M, 36, 36, a=a)
    assert np.allclose(out[outside == 0], 7.25, rtol=1e-14)
    # textbook values of the kernel: L(1/2) = 2a sin(pi/(2a)) / (pi^2/2 ...) written out for a = 3: 0.6079271
    assert po._lanczos(0.0, a) == 1.0 and po._lanczos(float(a), a) == 0.0 and po._lanczos(1.0, a) == 0.0
    assert po._lanczos(0.5, 3) == pytest.approx(3 * 1.0 * math.sin(math.pi / 6) / (math.pi ** 2 / 4), rel=1e-15)
    assert po._lanczos(0.5, 3) == pytest.approx(0.6079271018540267, rel=1e-12)


def test_resample_band_limited_wave_subpixel_shift():
    """A slowly varying sinusoid sampled off-grid: Lanczos-3 reproduces the analytic value to a few 1e-3."""
    y, x = np.mgrid[0:64, 0:64].astype(np.float64)
    f = lambda xx, yy: np.sin(2 * np.pi * xx / 23.0) * np.cos(2 * np.pi * yy / 31.0)
    M = [0.3, 1.0, 0.0, 0.45, 0.0, 1.0]
    out, outside = po.resample_affine(f(x, y), M, 60, 60, a=3)
    ok = outside == 0
    exact = f(x[:60, :60] + 0.3, y[:60, :60] + 0.45)
    assert np.max(np.abs(out[ok] - exact[ok])) < 6e-3
    assert np.max(np.abs(out[ok] - f(x[:60, :60], y[:60, :60])[ok])) > 0.05     # and it is not the unshifted image


def test_resample_mask_threshold():
    mask = np.zeros((20, 20), dtype=np.uint8)
    mask[10, 10] = 1
    out = po.resample_mask_affine(mask, IDENT, 20, 20)
    assert out[10, 10] == 2 and out[10, 11] == 1 and out[9, 10] == 1
    assert out[0, 0] == 2 and out[5, 5] == 1                  # outside -> bad, clean interior -> good
    # half-pixel shift in x: the bad pixel spreads L(0.5) = 0.608 > 0.3 onto both neighbours, the next ones get
    # L(1.5) = -0.135 < 0.3
    out = po.resample_mask_affine(mask, [0.5, 1.0, 0.0, 0.0, 0.0, 1.0], 20, 20)
    assert out[10, 9] == 2 and out[10, 10] == 2 and out[10, 8] == 1 and out[10, 11] == 1
