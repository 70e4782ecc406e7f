"""Seeded synthetic DECam-like star-field pairs (inputs only; none of the method's arithmetic).

These stand in for the paper's real DESIRT-2025A DECam exposures (§4.2), which
are not available.  Shapes, star counts, flux law, PSFs, sky and masks follow BASELINE.json
`configs[0..4]`; the items the configs leave open follow SURVEY.md §8(d) and are listed in
DESIGN.md ("Input recipe").

This module is the ONE piece shared by the CPU oracle's tests and the CUDA path's tests/bench.
It only draws random numbers and renders star profiles; it knows nothing about the delta-basis
fit, the normal equations or the FFTs.

Conventions: images are (H, W) float64, row-major, x fastest.  mask is uint8, nonzero = excluded.
"""
from __future__ import annotations

import dataclasses
import math
from typing import Callable, Optional

import numpy as np

__all__ = ["Config", "CONFIGS", "make_pair", "make_exposure_pair", "white_noise_pair", "Pair"]


@dataclasses.dataclass(frozen=True)
class Config:
    name: str
    H: int
    W: int
    w: int
    DK: int
    DB: int
    seed: int
    n_stars: int
    flux_lo: float
    flux_hi: float
    sky0: float
    read_noise: float
    border: int

    @property
    def L(self) -> int:
        return (2 * self.w + 1) ** 2

    @property
    def N(self) -> int:
        return self.L * (self.DK + 1) * (self.DK + 2) // 2 + (self.DB + 1) * (self.DB + 2) // 2

    @property
    def sky_rms(self) -> float:
        """sigma_sky = sqrt(sky_mean + RN^2) (gain 1 e-/ADU); the unit of the D tolerance."""
        return math.sqrt(self.sky0 + self.read_noise ** 2)


CONFIGS = {
    "tiny": Config("tiny", 64, 64, 2, 0, 0, 1001, 20, 1e3, 1e5, 100.0, 5.0, 2),
    "small": Config("small", 256, 256, 3, 1, 1, 1002, 150, 1e3, 1e6, 500.0, 5.0, 3),
    "mid": Config("mid", 1024, 1024, 4, 2, 2, 1003, 1000, 1e3, 1e6, 1000.0, 5.0, 4),
    "full": Config("full", 2048, 4096, 5, 2, 2, 1004, 3000, 1e3, 1e6, 1500.0, 6.0, 6),
    # the physical DECam orientation (2048 columns x 4096 rows); parity case only
    "full_t": Config("full_t", 4096, 2048, 5, 2, 2, 1005, 3000, 1e3, 1e6, 1500.0, 6.0, 6),
}


@dataclasses.dataclass
class Pair:
    cfg: Config
    R: np.ndarray
    S: np.ndarray
    mask: np.ndarray
    sky_rms: float


def _powerlaw_fluxes(rng, n, lo, hi):
    # inverse CDF of dN/dF ~ F^-2.5 on [lo, hi]
    u = rng.random(n)
    a, b = lo ** -1.5, hi ** -1.5
    return (a - u * (a - b)) ** (-1.0 / 1.5)


def _gauss(dx, dy, sigma):
    return np.exp(-(dx * dx + dy * dy) / (2.0 * sigma * sigma)) / (2.0 * math.pi * sigma * sigma)


def _moffat_r2(r2, fwhm, beta):
    alpha = fwhm / (2.0 * math.sqrt(2.0 ** (1.0 / beta) - 1.0))
    return (beta - 1.0) / (math.pi * alpha * alpha) * (1.0 + r2 / (alpha * alpha)) ** (-beta)


def _render(H, W, xs, ys, fluxes, half, profile: Callable):
    """Add point-sampled profiles (pixel-centre sampling) on stamps of half-size `half`."""
    img = np.zeros((H, W), dtype=np.float64)
    for i in range(len(xs)):
        cx, cy = xs[i], ys[i]
        x0, x1 = max(0, int(math.floor(cx)) - half), min(W, int(math.floor(cx)) + half + 1)
        y0, y1 = max(0, int(math.floor(cy)) - half), min(H, int(math.floor(cy)) + half + 1)
        if x1 <= x0 or y1 <= y0:
            continue
        dx = np.arange(x0, x1, dtype=np.float64)[None, :] - cx
        dy = np.arange(y0, y1, dtype=np.float64)[:, None] - cy
        img[y0:y1, x0:x1] += fluxes[i] * profile(i, dx, dy)
    return img


def _elliptical_moffat(fwhm, beta, e, theta):
    def prof(dx, dy):
        c, s = math.cos(theta), math.sin(theta)
        xp = c * dx + s * dy
        yp = -s * dx + c * dy
        r2 = xp * xp / (1.0 - e) + yp * yp * (1.0 - e)
        return _moffat_r2(r2, fwhm, beta)
    return prof


def make_pair(name: str, seed: Optional[int] = None, force_saturated: int = 0,
              sky0: Optional[float] = None, fwhm_s: Optional[float] = None) -> Pair:
    """One reference/science pair of BASELINE.json configs[0..3] (recipe: SURVEY.md §8(d))."""
    cfg = CONFIGS[name]
    if sky0 is not None:
        cfg = dataclasses.replace(cfg, sky0=float(sky0))
    rng = np.random.default_rng(cfg.seed if seed is None else seed)
    H, W = cfg.H, cfg.W
    xs = rng.random(cfg.n_stars) * W
    ys = rng.random(cfg.n_stars) * H
    fl = _powerlaw_fluxes(rng, cfg.n_stars, cfg.flux_lo, cfg.flux_hi)
    if force_saturated:
        bright = [2e6, 3e6, 5e6, 4e6, 6e6][:force_saturated]
        fl[: len(bright)] = bright
        # keep the forced stars away from the border so their cores are inside the frame
        xs[: len(bright)] = W * (0.25 + 0.5 * rng.random(len(bright)))
        ys[: len(bright)] = H * (0.25 + 0.5 * rng.random(len(bright)))
    xi = (2.0 * np.arange(W) + 1.0 - W) / W
    eta = (2.0 * np.arange(H) + 1.0 - H) / H
    XI, ETA = xi[None, :], eta[:, None]
    base = name.split("_")[0]

    if base == "tiny":
        fw = 3.0
        sr = fw / 2.3548
        ss = math.sqrt(sr * sr + 0.8 * 0.8)
        half = int(10 * fw)
        TR = _render(H, W, xs, ys, fl, half, lambda i, dx, dy: _gauss(dx, dy, sr))
        TS = _render(H, W, xs + 0.3, ys - 0.2, fl, half, lambda i, dx, dy: _gauss(dx, dy, ss))
        sky = np.full((H, W), cfg.sky0)
        sky_r = 0.0
    elif base == "small":
        fw = 3.5
        sr = fw / 2.3548
        half = int(10 * fw)
        sk = 0.6 + 0.6 * xs / W
        TR = _render(H, W, xs, ys, fl, half, lambda i, dx, dy: _gauss(dx, dy, sr))
        TS = _render(H, W, xs, ys, fl, half,
                     lambda i, dx, dy: _gauss(dx, dy, math.sqrt(sr * sr + sk[i] ** 2)))
        sky = cfg.sky0 + 50.0 * (np.arange(W, dtype=np.float64)[None, :] / W) + np.zeros((H, 1))
        sky_r = cfg.sky0
    elif base == "mid":
        from scipy.ndimage import gaussian_filter
        fw, beta = 4.0, 3.0
        half = int(10 * fw)
        sk = 0.8 + 0.3 * xs / W + 0.2 * ys / H
        TR = _render(H, W, xs, ys, fl, half,
                     lambda i, dx, dy: _moffat_r2(dx * dx + dy * dy, fw, beta))

        def prof_s(i, dx, dy):
            st = _moffat_r2(dx * dx + dy * dy, fw, beta)
            return gaussian_filter(st, sk[i], mode="constant")
        TS = _render(H, W, xs + 0.25, ys + 0.4, fl, half, prof_s)
        # 20 transients of 5e3 ADU in S only, S's local PSF
        nt = 20
        tx, ty = rng.random(nt) * W, rng.random(nt) * H
        tk = 0.8 + 0.3 * tx / W + 0.2 * ty / H

        def prof_t(i, dx, dy):
            st = _moffat_r2(dx * dx + dy * dy, fw, beta)
            return gaussian_filter(st, tk[i], mode="constant")
        TS += _render(H, W, tx, ty, np.full(nt, 5e3), half, prof_t)
        sky = cfg.sky0 + 80 * XI + 50 * ETA + 40 * XI ** 2 - 30 * XI * ETA + 20 * ETA ** 2
        sky_r = cfg.sky0
    elif base == "full":
        beta, fw_r = 2.5, 4.0
        fw_s = 5.0 if fwhm_s is None else float(fwhm_s)
        half = int(10 * fw_r)
        emax = 0.1
        ee = emax * xs / W
        th = math.pi * ys / H
        TR = _render(H, W, xs, ys, fl, half,
                     lambda i, dx, dy: _elliptical_moffat(fw_r, beta, ee[i], th[i])(dx, dy))
        TS = _render(H, W, xs, ys, fl, half,
                     lambda i, dx, dy: _elliptical_moffat(fw_s, beta, ee[i], th[i])(dx, dy))
        nt = 50
        tx, ty = rng.random(nt) * W, rng.random(nt) * H
        te, tt = emax * tx / W, math.pi * ty / H
        TS += _render(H, W, tx, ty, np.full(nt, 5e3), half,
                      lambda i, dx, dy: _elliptical_moffat(fw_s, beta, te[i], tt[i])(dx, dy))
        s0 = cfg.sky0
        sky = s0 + (120 * XI + 80 * ETA + 60 * XI ** 2 - 40 * XI * ETA + 30 * ETA ** 2) * (s0 / 1500.0)
        sky_r = s0
    else:
        raise KeyError(name)

    rn = cfg.read_noise
    R = rng.poisson(TR + sky_r).astype(np.float64) - sky_r + rng.normal(0.0, rn, (H, W))
    S = rng.poisson(TS + sky).astype(np.float64) + rng.normal(0.0, rn, (H, W))
    mask = np.zeros((H, W), dtype=np.uint8)
    b = cfg.border
    mask[:b, :] = 1
    mask[-b:, :] = 1
    mask[:, :b] = 1
    mask[:, -b:] = 1
    mask[(R + sky_r) > 6e4] = 1
    mask[S > 6e4] = 1
    return Pair(cfg, np.ascontiguousarray(R), np.ascontiguousarray(S), mask, cfg.sky_rms)


def make_exposure_pair(k: int) -> Pair:
    """CCD k of the 60-CCD exposure batch (BASELINE.json configs[4]): seed 2000+k,
    sky level ~ U[800,3000] ADU, science FWHM ~ U[3.5,6] px, reference FWHM fixed 4 px."""
    r = np.random.default_rng(900000 + k)
    return make_pair("full", seed=2000 + k, sky0=r.uniform(800.0, 3000.0),
                     fwhm_s=r.uniform(3.5, 6.0))


def white_noise_pair(H: int, W: int, seed: int, amp: float = 100.0):
    """Plain white-noise image(s) for exact-recovery pins and FFT checks (no star field)."""
    rng = np.random.default_rng(seed)
    return amp * rng.standard_normal((H, W)), amp * rng.standard_normal((H, W))
