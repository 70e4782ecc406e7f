"""CPU ORACLE for the two steps that follow SFFT differencing -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline legs may import this module.
It shares no code with the CUDA path and does not import the package.  Plain numpy loops, float64.

(1) Multi-template combination -- PAPER.md:158 (§2.3.2): "For multi-exposure templates, the science
    image is differenced against each individual template exposure, producing N_TEMP difference
    images per science exposure.  All difference images are subsequently normalized to a common
    photometric zero point (Section 2.3.1) and median-combined to produce a single final difference
    image"; N_TEMP "a tunable parameter with a default of 5" (§2.1.1).
    Definition written out: out[y,x] = median_k( scale_k * D_k[y,x] ), scale_k the flux factor that
    brings image k to the common zero point (scale_k = 10^(0.4 (zp_ref - zp_k))).
    Reading M1 (paper silent): for an even number of images the median is the mean of the two
    middle values (the usual convention; the default N_TEMP = 5 is odd).
    Reading M2 (paper silent): a NaN in any of the images makes the combined pixel NaN (what
    numpy.median does; a resampled template flags its missing pixels this way).

(2) Monte-Carlo limiting flux -- PAPER.md:164 (§2.3.3): "We measure aperture fluxes at 1024 randomly
    selected background positions using the same aperture definition, and deriving the 5 sigma
    threshold from their standard deviation, converted to magnitudes with the corresponding zero
    point"; aperture "0.6731 x FWHM" (§2.3.1).
    Readings (paper silent): L1 the aperture is the hard-edged disc of pixels whose centres lie within
    `radius` of the (real-valued) position, pixel (y,x) centred at integer coordinates; L2 a position
    is a "background position" when its disc lies inside the frame and touches no masked pixel --
    other positions are dropped (flux NaN); L3 the standard deviation is the population one
    (divide by the number of kept apertures); L4 the positions are inputs (the random draw is the
    caller's), so both sides see the same ones; L5 m_lim = zp - 2.5 log10(5 sigma).

(3) Multi-template MODE, the whole chain of (1) -- PAPER.md:158 (§2.3.2) with N_TEMP of PAPER.md:94:
    multi_template_difference = N_TEMP runs of the differencing oracle (oracle/sfft_oracle.py, one per
    template exposure, all against the same science image), then (1).  Reading MT1 (paper silent on
    which pixels enter each fit): one common mask -- the union of the science and template data-quality
    masks (PAPER.md:162 treats a pixel as bad when it is flagged "in either the science or template
    images") -- is used in all N_TEMP fits; a list of per-template masks is accepted too.

(4) Three-channel stamps for the real-bogus classifier -- PAPER.md:168 (§2.3.4): "the classifier takes
    as input a set of three-channel image stamps -- consisting of the science image, template image,
    and their difference -- centered on the candidate position".  The paper gives neither the stamp
    size nor an edge rule; readings: ST1 channel order (science, template, difference), as listed;
    ST2 the stamp is size x size pixels, its centre pixel (index size//2 along each axis) is the pixel
    nearest the position, (floor(x + 1/2), floor(y + 1/2)), pixel centres at integer coordinates;
    ST3 pixels outside the frame are 0; ST4 a non-finite position gives an all-NaN stamp.

Pins (tests/test_post_pins.py): statistics.median on small stacks, permutation and scale
invariance, known order statistics; Gauss circle lattice counts N(r) for the disc, a constant image
(flux = c N(r), sigma = 0), a linear ramp (flux = N(r) * value at the centre for integer centres),
white noise (sigma ~ sigma_pix sqrt N(r)), masked / out-of-frame positions dropped.
"""
from __future__ import annotations

import math

import numpy as np


def median_combine(Ds, scales):
    """out = median over k of scales[k] * Ds[k], element by element (sort, take the middle)."""
    stack = np.stack([np.asarray(D, dtype=np.float64) * float(s) for D, s in zip(Ds, scales)], axis=0)
    n = stack.shape[0]
    srt = np.sort(stack, axis=0)
    out = srt[n // 2].copy() if n % 2 == 1 else 0.5 * (srt[n // 2 - 1] + srt[n // 2])
    out[np.isnan(stack).any(axis=0)] = np.nan      # reading M2: a NaN in any image makes the pixel NaN
    return out


def aperture_flux(D, mask, x0, y0, radius):
    """Sum of D over the pixels whose centres lie within `radius` of (x0, y0); NaN if the disc
    leaves the frame or touches a masked pixel (readings L1, L2).  Explicit loops."""
    H, W = D.shape
    r2 = radius * radius
    if not (math.isfinite(x0) and math.isfinite(y0)):
        return float("nan")                        # reading L2: not a position inside the frame
    ylo, yhi = int(math.ceil(y0 - radius)), int(math.floor(y0 + radius))
    xlo, xhi = int(math.ceil(x0 - radius)), int(math.floor(x0 + radius))
    if ylo < 0 or xlo < 0 or yhi > H - 1 or xhi > W - 1:
        return float("nan")
    tot = 0.0
    for y in range(ylo, yhi + 1):
        for x in range(xlo, xhi + 1):
            if (x - x0) ** 2 + (y - y0) ** 2 <= r2:
                if mask is not None and mask[y, x]:
                    return float("nan")
                tot += float(D[y, x])
    return tot


def aperture_stats(D, mask, xs, ys, radius):
    """Fluxes at the given positions and (count, mean, population sigma) of the kept ones."""
    flux = np.array([aperture_flux(D, mask, float(x), float(y), radius) for x, y in zip(xs, ys)])
    kept = flux[~np.isnan(flux)]
    n = kept.size
    if n == 0:
        return flux, (0, float("nan"), float("nan"))
    mean = float(np.sum(kept) / n)
    sigma = float(math.sqrt(np.sum((kept - mean) ** 2) / n))
    return flux, (n, mean, sigma)


def limiting_magnitude(sigma, zero_point):
    """m_lim = zp - 2.5 log10(5 sigma)  (reading L5)."""
    return zero_point - 2.5 * math.log10(5.0 * sigma)


def multi_template_difference(Rs, S, masks, w, DK, DB, scales, workers=1):
    """(D_final, [D_k], [c_k]): one differencing per template R_k against the same S,
    D_final = median_k(scales[k] * D_k).  `masks`: one common mask (reading MT1), None, or a list."""
    from oracle import sfft_oracle as orc
    if masks is None or isinstance(masks, np.ndarray):
        masks = [masks] * len(Rs)
    Ds, cs = [], []
    for R, m in zip(Rs, masks):
        _, _, c, D = orc.sfft_difference(R, S, m, w, DK, DB, workers=workers, fourier_subtract=True)
        Ds.append(D)
        cs.append(c)
    return median_combine(Ds, scales), Ds, cs


def cut_stamps(S, R, D, xs, ys, size):
    """[n, 3, size, size] stamps (science, template, difference) centred on the positions
    (readings ST1-ST4).  Explicit loops."""
    H, W = S.shape
    n = len(xs)
    out = np.zeros((n, 3, size, size))
    half = size // 2
    for k in range(n):
        x, y = float(xs[k]), float(ys[k])
        if not (math.isfinite(x) and math.isfinite(y)):
            out[k] = np.nan
            continue
        cx, cy = math.floor(x + 0.5), math.floor(y + 0.5)
        for ch, img in enumerate((S, R, D)):
            for j in range(size):
                for i in range(size):
                    yy, xx = cy - half + j, cx - half + i
                    if 0 <= yy < H and 0 <= xx < W:
                        out[k, ch, j, i] = img[yy, xx]
    return out


# --------------------------------------------------------------------------- resampling (NEXT-4)
# PAPER.md:156 (§2.3.2): "We first reproject the new science image onto the WCS of the corresponding
# template image(s) using SWARP ... ensuring pixel-level alignment"; PAPER.md:96, 118 (§2.1.1): archival
# exposures and their data-quality masks are "resampled onto the expected WCS of the target CCD";
# "the resampled ood images are discretized using an empirical threshold of 0.3: pixels with values
# above 0.3 are flagged as bad (set to 2^1), and others are flagged as good (set to 2^0)".
# The paper gives neither the interpolant nor a WCS; readings:
#   R1 the pixel map is an affine one, x_in = M0 + M1 x_out + M2 y_out, y_in = M3 + M4 x_out + M5 y_out
#      (a synthetic stand-in for the WCS pair; pixel centres at integer coordinates);
#   R2 the interpolant is the separable Lanczos kernel of order a (SWarp's default resampling is
#      LANCZOS3): L(t) = sinc(t) sinc(t/a) for |t| < a, else 0, taps at floor(x_in) - a + 1 .. + a;
#   R3 the 2a x 2a weights are divided by their sum (a constant image stays constant); no Jacobian
#      flux factor is applied;
#   R4 an output pixel whose taps leave the input frame is set to 0 and reported as outside;
#   R5 masks: the 0/1 bad indicator is interpolated with the same weights, value > 0.3 -> 2 (bad),
#      else 1 (good); outside pixels are bad.


def _lanczos(t, a):
    t = abs(t)
    if t >= a:
        return 0.0
    if t == 0.0:
        return 1.0
    if t == math.floor(t):
        return 0.0          # sinc vanishes at the non-zero integers (exactly, not to rounding)
    pt = math.pi * t
    return a * math.sin(pt) * math.sin(pt / a) / (pt * pt)


def resample_affine(img, M, Hout, Wout, a=3):
    """(out, outside): Lanczos-a resampling of `img` through the affine map M (readings R1-R4)."""
    Hin, Win = img.shape
    out = np.zeros((Hout, Wout))
    outside = np.zeros((Hout, Wout), dtype=np.uint8)
    for yo in range(Hout):
        for xo in range(Wout):
            xi = M[0] + M[1] * xo + M[2] * yo
            yi = M[3] + M[4] * xo + M[5] * yo
            x0, y0 = math.floor(xi), math.floor(yi)
            if x0 - a + 1 < 0 or y0 - a + 1 < 0 or x0 + a > Win - 1 or y0 + a > Hin - 1:
                outside[yo, xo] = 1
                continue
            wx = [_lanczos(xi - (x0 - a + 1 + k), a) for k in range(2 * a)]
            wy = [_lanczos(yi - (y0 - a + 1 + k), a) for k in range(2 * a)]
            acc = 0.0
            for j in range(2 * a):
                row = 0.0
                for k in range(2 * a):
                    row += wx[k] * float(img[y0 - a + 1 + j, x0 - a + 1 + k])
                acc += wy[j] * row
            out[yo, xo] = acc / (sum(wx) * sum(wy))
    return out, outside


def resample_mask_affine(mask, M, Hout, Wout, a=3, threshold=0.3):
    """Resampled data-quality mask: 2 = bad, 1 = good (readings R4, R5)."""
    val, outside = resample_affine((np.asarray(mask) != 0).astype(np.float64), M, Hout, Wout, a)
    return np.where((val > threshold) | (outside != 0), 2, 1).astype(np.uint8)
