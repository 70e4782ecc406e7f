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


# --------------------------------------------------------------------------- stamps
def test_stamps_hand_written_values():
    """5x6 images with value 10 y + x (science), 100 + that (template), -that (difference): stamps
    written out by hand for an interior, a corner and an off-frame position (readings ST1-ST3)."""
    H, W = 5, 6
    base = np.array([[10.0 * y + x for x in range(W)] for y in range(H)])
    S, R, D = base, 100.0 + base, -base
    st = po.cut_stamps(S, R, D, [2.0, 0.0, 5.4, -3.0], [2.0, 0.0, 4.2, 1.0], 3)
    assert st.shape == (4, 3, 3, 3)
    assert st[0, 0].tolist() == [[11, 12, 13], [21, 22, 23], [31, 32, 33]]
    assert st[0, 1].tolist() == [[111, 112, 113], [121, 122, 123], [131, 132, 133]]
    assert st[0, 2].tolist() == [[-11, -12, -13], [-21, -22, -23], [-31, -32, -33]]
    assert st[1, 0].tolist() == [[0, 0, 0], [0, 0, 1], [0, 10, 11]]          # top-left corner: zero fill
    assert st[2, 0].tolist() == [[34, 35, 0], [44, 45, 0], [0, 0, 0]]        # (5.4, 4.2) -> pixel (5, 4)
    assert st[3].tolist() == np.zeros((3, 3, 3)).tolist()                    # wholly outside the frame


def test_stamps_rounding_even_size_and_nonfinite():
    H, W = 8, 8
    S = np.arange(64.0).reshape(H, W)
    # nearest pixel: floor(x + 1/2) -- 2.5 -> 3, 2.49 -> 2, -0.5 -> 0, -0.51 -> -1
    st = po.cut_stamps(S, S, S, [2.5, 2.49, -0.5, -0.51], [3.0, 3.0, 3.0, 3.0], 1)
    assert st[:, 0, 0, 0].tolist() == [27.0, 26.0, 24.0, 0.0]
    # even size: the centre pixel has index size//2, so the stamp starts size//2 before it
    st = po.cut_stamps(S, S, S, [4.0], [4.0], 4)
    assert st[0, 0, 2, 2] == S[4, 4] and st[0, 0, 0, 0] == S[2, 2] and st[0, 0, 3, 3] == S[5, 5]
    st = po.cut_stamps(S, S, S, [float("nan"), float("inf")], [1.0, 1.0], 3)
    assert np.isnan(st).all()


# ------------------------------------------------------------- multi-template mode
def _mt_pair(seed, H=32, W=32):
    rng = np.random.default_rng(seed)
    R = 50.0 * rng.standard_normal((H, W)) + 400.0 * (rng.random((H, W)) > 0.97)
    S = 0.8 * np.roll(R, (1, -1), (0, 1)) + 5.0 * rng.standard_normal((H, W)) + 120.0
    mask = (rng.random((H, W)) < 0.04).astype(np.uint8)
    return R, S, mask


def test_multi_template_identical_templates_equal_the_single_difference():
    from oracle import sfft_oracle as orc
    R, S, mask = _mt_pair(1)
    _, _, _, D1 = orc.sfft_difference(R, S, mask, 1, 1, 1)
    Dm, Ds, cs = po.multi_template_difference([R] * 5, S, mask, 1, 1, 1, [1.0] * 5)
    assert len(Ds) == 5 and np.array_equal(Dm, D1)


def test_multi_template_permutation_invariance_and_outlier_rejection():
    rng = np.random.default_rng(2)
    R, S, mask = _mt_pair(2)
    # five different templates (independent noise realisations of the same field)
    Rs = [R + 3.0 * rng.standard_normal(R.shape) for _ in range(5)]
    sc = [1.0, 1.1, 0.9, 1.05, 0.95]
    Dm, Ds, _ = po.multi_template_difference(Rs, S, mask, 1, 0, 0, sc)
    perm = [3, 0, 4, 1, 2]
    Dp, _, _ = po.multi_template_difference([Rs[i] for i in perm], S, mask, 1, 0, 0, [sc[i] for i in perm])
    assert np.array_equal(Dm, Dp)
    # the result is, pixel by pixel, one of the scaled individual differences (odd count)
    stack = np.stack([s * D for s, D in zip(sc, Ds)])
    assert np.all(np.any(stack == Dm[None], axis=0))
    # four identical templates and one carrying an artefact: at least three of the five values of
    # every pixel agree exactly, so the artefact never reaches the median
    Rbad = R.copy()
    Rbad[10:14, 10:14] += 5000.0
    Dclean, _, _ = po.multi_template_difference([R] * 5, S, mask, 1, 0, 0, [1.0] * 5)
    for pos in range(5):
        Rs2 = [R] * 5
        Rs2[pos] = Rbad
        Dout, Ds2, _ = po.multi_template_difference(Rs2, S, mask, 1, 0, 0, [1.0] * 5)
        assert np.array_equal(Dout, Dclean)
        assert np.max(np.abs(Ds2[pos] - Dclean)) > 100.0      # the artefact is in that one difference


def test_multi_template_per_template_masks_and_common_mask_agree_when_equal():
    R, S, mask = _mt_pair(3)
    a, _, _ = po.multi_template_difference([R, 1.01 * R, 0.99 * R], S, mask, 1, 0, 0, [1.0, 1.0, 1.0])
    b, _, _ = po.multi_template_difference([R, 1.01 * R, 0.99 * R], S, [mask, mask, mask], 1, 0, 0, [1.0, 1.0, 1.0])
    assert np.array_equal(a, b)
