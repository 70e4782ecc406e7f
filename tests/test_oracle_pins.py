"""Pins for the CPU oracle (oracle/sfft_oracle.py) against things other than itself:
brute force, closed forms, invariants, library routines on special cases, exact recovery.
Numbering P1..P18 follows SURVEY.md §8(c) "What pins each part".  CPU only.
"""
import os
from fractions import Fraction

import numpy as np
import pytest
import scipy.signal

from oracle import sfft_oracle as orc
from paper_2603_08593_b200 import synth

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def _rand_case(H, W, seed, masked=True, border=0):
    rng = np.random.default_rng(seed)
    R = 50.0 * rng.standard_normal((H, W)) + 200.0 * (rng.random((H, W)) > 0.97)
    S = 40.0 * rng.standard_normal((H, W)) + 300.0
    mask = None
    if masked:
        mask = (rng.random((H, W)) < 0.08).astype(np.uint8)
        if border:
            mask[:border] = 1
            mask[-border:] = 1
            mask[:, :border] = 1
            mask[:, -border:] = 1
    return R, S, mask


# ------------------------------------------------------------------ conventions

def test_conventions_orders_and_counts():
    assert orc.monomials(2) == [(0, 0), (1, 0), (0, 1), (2, 0), (1, 1), (0, 2)]
    sh = orc.shifts(2)
    assert sh[0] == (-2, -2) and sh[1] == (-1, -2) and sh[-1] == (2, 2)
    for s, (u, v) in enumerate(sh):
        assert s == (v + 2) * 5 + (u + 2)
    # N at the four configs (BASELINE.json north_star / SURVEY 8.0 size table)
    assert [orc.num_coeffs(2, 0, 0), orc.num_coeffs(3, 1, 1), orc.num_coeffs(4, 2, 2),
            orc.num_coeffs(5, 2, 2)] == [26, 150, 492, 732]
    xi, eta = orc.coords(8, 4)
    assert np.allclose(xi, [-0.75, -0.25, 0.25, 0.75]) and eta[0] == -7 / 8 and eta[-1] == 7 / 8


# ------------------------------------------------------------------ A, b

@pytest.mark.parametrize("H,W,w,DK,DB,masked", [
    (24, 40, 2, 1, 2, True), (32, 16, 1, 2, 1, True), (20, 28, 2, 0, 0, False)])
def test_P1_bruteforce_equals_fft_route(H, W, w, DK, DB, masked):
    R, S, mask = _rand_case(H, W, 7 + H, masked)
    A1, b1 = orc.build_system_bruteforce(R, S, mask, w, DK, DB)
    A2, b2 = orc.build_system_fft(R, S, mask, w, DK, DB)
    assert np.max(np.abs(A1 - A2)) <= 1e-13 * np.max(np.abs(A1))
    assert np.max(np.abs(b1 - b2)) <= 1e-13 * np.max(np.abs(b1))


def test_P1_tiny_config_bruteforce_equals_fft_route():
    pr = synth.make_pair("tiny")
    c = pr.cfg
    A1, b1 = orc.build_system_bruteforce(pr.R, pr.S, pr.mask, c.w, c.DK, c.DB)
    A2, b2 = orc.build_system_fft(pr.R, pr.S, pr.mask, c.w, c.DK, c.DB)
    assert A1.shape == (26, 26)
    assert np.max(np.abs(A1 - A2)) <= 1e-13 * np.max(np.abs(A1))
    assert np.max(np.abs(b1 - b2)) <= 1e-13 * np.max(np.abs(b1))


def test_single_entry_sums_match_bruteforce():
    R, S, mask = _rand_case(24, 40, 3)
    w, DK, DB = 2, 1, 1
    A, b = orc.build_system_bruteforce(R, S, mask, w, DK, DB)
    N = A.shape[0]
    rng = np.random.default_rng(0)
    for _ in range(25):
        i, j = rng.integers(0, N, 2)
        assert abs(orc.normal_entry(R, S, mask, w, DK, DB, i, j) - A[i, j]) <= 1e-12 * np.abs(A).max()
    for i in (0, 7, N - 1, N - 3):
        assert abs(orc.normal_entry(R, S, mask, w, DK, DB, i) - b[i]) <= 1e-12 * np.abs(b).max()


def test_P2_symmetric_psd_and_P3_block_toeplitz():
    H, W, w, DK, DB = 24, 32, 2, 1, 1
    R, S, mask = _rand_case(H, W, 11)
    A, b = orc.build_system_fft(R, S, mask, w, DK, DB)
    assert np.array_equal(A, A.T)
    ev = np.linalg.eigvalsh(A)
    assert ev.min() >= -1e-9 * ev.max()
    L = (2 * w + 1) ** 2
    sh = orc.shifts(w)
    TK = 3
    m = (mask == 0).astype(float)
    xi, eta = orc.coords(H, W)
    for t, (p, q) in enumerate(orc.monomials(DK)):
        blk = A[t * L:(t + 1) * L, t * L:(t + 1) * L]
        d = np.diag(blk)
        # diag constant inside a polynomial block and equal to sum R~_t^2
        assert np.ptp(d) <= 1e-12 * abs(d[0])
        Rt = m * np.multiply.outer(eta ** q, xi ** p) * R
        assert abs(d[0] - np.sum(Rt * Rt)) <= 1e-12 * abs(d[0])
    # entries depend only on the shift difference
    for t in range(TK):
        for t2 in range(TK):
            seen = {}
            blk = A[t * L:(t + 1) * L, t2 * L:(t2 + 1) * L]
            for s, (u, v) in enumerate(sh):
                for s2, (u2, v2) in enumerate(sh):
                    key = (u - u2, v - v2)
                    if key in seen:
                        assert abs(seen[key] - blk[s, s2]) <= 1e-12 * np.abs(A).max()
                    else:
                        seen[key] = blk[s, s2]


def _golden_moments():
    tab = {}
    with open(os.path.join(GOLDEN, "bb_moments.txt")) as f:
        for line in f:
            if line.startswith("#"):
                continue
            n, a, num, den, _ = line.split()
            tab[(int(n), int(a))] = Fraction(int(num), int(den))
    return tab


@pytest.mark.parametrize("H,W,DB", [(16, 64, 2), (64, 16, 3), (256, 64, 2)])
def test_P4_background_block_closed_form(H, W, DB):
    """mask=NULL: A[B(p,q),B(p',q')] = mx(p+p';W) my(q+q';H), exact rationals from tests/golden."""
    tab = _golden_moments()
    R, S, _ = _rand_case(H, W, 5, masked=False)
    w, DK = 1, 0
    A, b = orc.build_system_fft(R, S, None, w, DK, DB)
    L = 9
    mono = orc.monomials(DB)
    for i, (p, q) in enumerate(mono):
        for j, (p2, q2) in enumerate(mono):
            exact = float(tab[(W, p + p2)] * tab[(H, q + q2)])
            got = A[L + i, L + j]
            assert abs(got - exact) <= 1e-12 * H * W, (p, q, p2, q2, got, exact)
    assert A[L, L] == H * W
    assert abs(A[L + 1, L + 1] - H * (W * W - 1) / (3 * W)) <= 1e-10
    assert abs(A[L + 2, L + 2] - W * (H * H - 1) / (3 * H)) <= 1e-10
    assert abs(A[L, L + 1]) <= 1e-9 and abs(A[L, L + 2]) <= 1e-9


def test_P5_rhs_background_zero_is_masked_sum():
    R, S, mask = _rand_case(24, 32, 2)
    A, b = orc.build_system_fft(R, S, mask, 2, 1, 1)
    assert abs(b[3 * 25] - np.sum(S[mask == 0])) <= 1e-12 * abs(b[3 * 25])
    assert A[3 * 25, 3 * 25] == np.sum(mask == 0)


def test_P6_bordered_maps_equal_zero_padded_library_correlation():
    """With a masked border >= w the circular maps equal scipy.signal.correlate2d (zero padded)
    on every lag used, so A's K-K block for DK=0 is a library cross-correlation (A7)."""
    H, W, w = 20, 24, 2
    R, S, mask = _rand_case(H, W, 9, masked=True, border=w)
    A, b = orc.build_system_fft(R, S, mask, w, 0, 0)
    Rm = (mask == 0) * R
    Sm = (mask == 0) * S
    full = scipy.signal.correlate2d(Rm, Rm, mode="full")  # full[dy+H-1, dx+W-1] = sum Rm(x+d) Rm(x)
    fullS = scipy.signal.correlate2d(Sm, Rm, mode="full")
    sh = orc.shifts(w)
    L = len(sh)
    for s, (u, v) in enumerate(sh):
        for s2, (u2, v2) in enumerate(sh):
            lib = full[(v - v2) + H - 1, (u - u2) + W - 1]
            assert abs(A[s, s2] - lib) <= 1e-12 * np.abs(A).max()
        assert abs(b[s] - fullS[v + H - 1, u + W - 1]) <= 1e-12 * np.abs(b).max()


def test_P7_linearity_scalings():
    R, S, mask = _rand_case(16, 24, 4)
    w, DK, DB = 1, 1, 1
    A, b = orc.build_system_fft(R, S, mask, w, DK, DB)
    A2, b2 = orc.build_system_fft(3.0 * R, 2.0 * S, mask, w, DK, DB)
    nK = 9 * 3
    assert np.allclose(A2[:nK, :nK], 9.0 * A[:nK, :nK], rtol=1e-13)
    assert np.allclose(A2[:nK, nK:], 3.0 * A[:nK, nK:], rtol=1e-12, atol=1e-9)
    assert np.allclose(A2[nK:, nK:], A[nK:, nK:], rtol=1e-13)
    assert np.allclose(b2[:nK], 6.0 * b[:nK], rtol=1e-12, atol=1e-7)
    assert np.allclose(b2[nK:], 2.0 * b[nK:], rtol=1e-13)


# ------------------------------------------------------------------ c

def test_P8_identity_and_P9_integer_shift():
    H, W, w, DK, DB = 32, 40, 2, 1, 1
    R, _ = synth.white_noise_pair(H, W, 1)
    L = 25
    for (u0, v0) in [(0, 0), (2, -1), (-2, 2)]:
        S = np.roll(R, shift=(v0, u0), axis=(0, 1))
        A, b = orc.build_system_fft(R, S, None, w, DK, DB)
        c = orc.solve(A, b)
        expect = np.zeros_like(c)
        expect[(v0 + w) * 5 + (u0 + w)] = 1.0      # constant term t=0, shift (u0,v0): A6 sign
        assert np.max(np.abs(c - expect)) <= 1e-10
        D = orc.subtract_rollsum(R, S, c, w, DK, DB)
        assert np.max(np.abs(D)) <= 1e-9 * np.max(np.abs(S))


def _random_truth(w, DK, DB, seed):
    rng = np.random.default_rng(seed)
    L = (2 * w + 1) ** 2
    TK = (DK + 1) * (DK + 2) // 2
    TB = (DB + 1) * (DB + 2) // 2
    c0 = np.zeros(L * TK + TB)
    sh = orc.shifts(w)
    base = np.array([np.exp(-((u - 0.3) ** 2 + (v + 0.2) ** 2) / (2 * 0.8 ** 2)) for (u, v) in sh])
    base /= base.sum()
    c0[:L] = base
    for t in range(1, TK):
        c0[t * L:(t + 1) * L] = 0.2 * base * rng.standard_normal(L)
    c0[L * TK:] = rng.standard_normal(TB) * 30.0
    c0[L * TK] = 100.0
    return c0


@pytest.mark.parametrize("H,W,w,DK,DB", [(48, 64, 2, 0, 0), (64, 48, 2, 2, 2), (40, 40, 3, 1, 2)])
def test_P10_exact_recovery_P11_optimality_P15_zero_residual(H, W, w, DK, DB):
    """S = M(R; c0) with mask=NULL and noisy R  =>  c = c0 to <= 1e-9 relative (north_star)."""
    R, _ = synth.white_noise_pair(H, W, 21)
    c0 = _random_truth(w, DK, DB, 3)
    S = orc.model_rollsum(R, c0, w, DK, DB)
    A, b = orc.build_system_fft(R, S, None, w, DK, DB)
    c = orc.solve(A, b)
    assert np.max(np.abs(c - c0)) <= 1e-9 * np.max(np.abs(c0))
    G, St = orc.design_matrix(R, S, None, w, DK, DB)
    assert np.max(np.abs(G.T @ (St - G @ c))) <= 1e-9 * np.max(np.abs(b))       # P11
    D = orc.subtract_rollsum(R, S, c, w, DK, DB)
    assert np.max(np.abs(D)) <= 1e-10 * np.max(np.abs(S))                       # P15


def test_P12_cholesky_equals_lstsq_and_P13_textbook_constant_kernel():
    pr = synth.make_pair("tiny")
    cfg = pr.cfg
    A, b = orc.build_system_fft(pr.R, pr.S, pr.mask, cfg.w, cfg.DK, cfg.DB)
    c = orc.solve(A, b)
    # P13: DK=DB=0 is plain linear regression on 25 shifted copies + a constant (Bramich 2008,
    # cited PAPER.md:40,387); built here without the oracle's helpers.
    m = (pr.mask == 0).astype(float)
    cols = [np.roll(m * pr.R, (v, u), (0, 1)).ravel() for v in range(-2, 3) for u in range(-2, 3)]
    cols.append(m.ravel())
    Gm = np.stack(cols, 1)
    c_ls = np.linalg.lstsq(Gm, (m * pr.S).ravel(), rcond=None)[0]
    assert np.max(np.abs(c - c_ls)) <= 1e-9 * np.max(np.abs(c_ls))
    # P12 on a spatially varying case
    R, S, mask = _rand_case(24, 32, 8)
    G, St = orc.design_matrix(R, S, mask, 1, 1, 1)
    A, b = orc.build_system_fft(R, S, mask, 1, 1, 1)
    c2 = orc.solve(A, b)
    c2_ls = np.linalg.lstsq(G, St, rcond=None)[0]
    assert np.max(np.abs(c2 - c2_ls)) <= 1e-9 * np.max(np.abs(c2_ls))


def test_nonpositive_definite_raises():
    R = np.zeros((16, 16))
    S = np.ones((16, 16))
    A, b = orc.build_system_fft(R, S, None, 1, 0, 0)
    with pytest.raises(np.linalg.LinAlgError):
        orc.solve(A, b)


# ------------------------------------------------------------------ D

def test_P14_rollsum_equals_fourier_route_and_pixel_samples():
    H, W, w, DK, DB = 32, 48, 2, 2, 1
    R, S, _ = _rand_case(H, W, 13, masked=False)
    c = _random_truth(w, DK, DB, 5)
    D1 = orc.subtract_rollsum(R, S, c, w, DK, DB)
    D2 = orc.subtract_fft(R, S, c, w, DK, DB)
    assert np.max(np.abs(D1 - D2)) <= 1e-12 * np.max(np.abs(D1))
    ys = np.array([0, 1, 31, 17, 5])
    xs = np.array([0, 47, 2, 23, 46])
    Dp = orc.subtract_at_pixels(R, S, c, w, DK, DB, ys, xs)
    assert np.max(np.abs(Dp - D1[ys, xs])) <= 1e-12 * np.max(np.abs(D1))


def test_P16_difference_invariant_under_coordinate_choice():
    """Any affine re-parametrisation of the polynomial coordinates spans the same space, so the
    fitted D is unchanged (A3).  The alternative basis (raw pixel indices) is built here."""
    H, W, w = 20, 24, 1
    R, S, mask = _rand_case(H, W, 17)
    DK = DB = 1
    A, b = orc.build_system_fft(R, S, mask, w, DK, DB)
    D = orc.subtract_rollsum(R, S, orc.solve(A, b), w, DK, DB)
    m = (mask == 0).astype(float)
    X, Y = np.meshgrid(np.arange(W, dtype=float), np.arange(H, dtype=float))
    polys = [np.ones((H, W)), X, Y]
    cols, cols_un = [], []
    for Pt in polys:
        for v in range(-w, w + 1):
            for u in range(-w, w + 1):
                cols.append(np.roll(m * Pt * R, (v, u), (0, 1)).ravel())
                cols_un.append(np.roll(Pt * R, (v, u), (0, 1)).ravel())
    for Pt in polys:
        cols.append((m * Pt).ravel())
        cols_un.append(Pt.ravel())
    c_alt = np.linalg.lstsq(np.stack(cols, 1), (m * S).ravel(), rcond=None)[0]
    D_alt = S - (np.stack(cols_un, 1) @ c_alt).reshape(H, W)
    assert np.max(np.abs(D - D_alt)) <= 1e-8 * np.max(np.abs(S))


def test_P17_P18_small_config_background_and_noise_level():
    pr = synth.make_pair("small")
    cfg = pr.cfg
    A, b, c, D = orc.sfft_difference(pr.R, pr.S, pr.mask, cfg.w, cfg.DK, cfg.DB)
    beta = c[-3:]
    # injected sky 500 + 50 x/W = 525 + 25 xi (+ half-pixel offset 50/(2W) absorbed below)
    assert abs(beta[0] - 525.0) < 2.0 and abs(beta[1] - 25.0) < 2.0 and abs(beta[2]) < 2.0
    good = D[pr.mask == 0]
    mad = 1.4826 * np.median(np.abs(good - np.median(good)))
    ksum2 = np.sum(c[:49] ** 2)
    pred = np.sqrt(cfg.sky0 + 25.0 + ksum2 * (cfg.sky0 + 25.0))
    assert 0.8 * pred < mad < 1.25 * pred


def test_O5_longdouble_referee_agrees():
    R, S, mask = _rand_case(32, 32, 23)
    A, b = orc.build_system_fft(R, S, mask, 2, 1, 1)
    Al, bl = orc.build_system_fft(R, S, mask, 2, 1, 1, dtype=np.longdouble)
    assert np.max(np.abs(A - Al.astype(np.float64))) <= 1e-14 * np.max(np.abs(A))
    assert np.max(np.abs(b - bl.astype(np.float64))) <= 1e-14 * np.max(np.abs(b))


# --------------------------------------------------------------------------- exact objective (NEXT-1)
def test_exact_objective_recovers_a_known_kernel_under_a_mask():
    """The literal objective (masked pixels dropped from the sum, images unmasked): S = M(R; c0) gives
    c = c0 to 1e-9 under a random 8 % mask + border -- which the input-masking reading A2 cannot (A2')."""
    H, W, w, DK, DB = 40, 48, 2, 1, 1
    R, _, mask = _rand_case(H, W, 21, masked=True, border=3)
    rng = np.random.default_rng(4)
    N = orc.num_coeffs(w, DK, DB)
    c0 = 0.1 * rng.standard_normal(N)
    c0[12] = 1.0
    c0[-3:] = [250.0, 10.0, -5.0]
    S = orc.model_rollsum(R, c0, w, DK, DB)
    A, b = orc.build_system_exact_bruteforce(R, S, mask, w, DK, DB)
    c = orc.solve(A, b)
    assert np.max(np.abs(c - c0)) <= 1e-9 * np.max(np.abs(c0))
    # the input-masking system does not recover it (reading A2')
    A2, b2 = orc.build_system_bruteforce(R, S, mask, w, DK, DB)
    assert np.max(np.abs(orc.solve(A2, b2) - c0)) > 1e-4 * np.max(np.abs(c0))


def test_exact_objective_equals_lstsq_on_unmasked_pixels_and_fft_route():
    H, W, w, DK, DB = 32, 40, 2, 1, 2
    R, S, mask = _rand_case(H, W, 22, masked=True, border=0)
    A, b = orc.build_system_exact_bruteforce(R, S, mask, w, DK, DB)
    G, St = orc.design_matrix(R, S, None, w, DK, DB)
    keep = mask.ravel() == 0
    c_ls = np.linalg.lstsq(G[keep], St[keep], rcond=None)[0]      # library QR/SVD on the plain definition
    assert np.max(np.abs(orc.solve(A, b) - c_ls)) <= 1e-9 * np.max(np.abs(c_ls))
    A2, b2 = orc.build_system_exact_fft(R, S, mask, w, DK, DB)    # unmasked Fourier route minus rank-one terms
    assert np.max(np.abs(A2 - A)) <= 1e-12 * np.max(np.abs(A))
    assert np.max(np.abs(b2 - b)) <= 1e-12 * np.max(np.abs(b))
    # sampled entries by direct sums over the unmasked pixels
    for (i, j) in [(0, 0), (3, 40), (60, 7), (A.shape[0] - 1, 5), (A.shape[0] - 2, A.shape[0] - 1)]:
        assert orc.exact_entry(R, S, mask, w, DK, DB, i, j) == pytest.approx(A[i, j], rel=1e-12, abs=1e-9 * np.max(np.abs(A)))
    assert orc.exact_entry(R, S, mask, w, DK, DB, 11) == pytest.approx(b[11], rel=1e-12)
    # mask = None: both objectives coincide
    A3, b3 = orc.build_system_exact_bruteforce(R, S, None, w, DK, DB)
    A4, b4 = orc.build_system_bruteforce(R, S, None, w, DK, DB)
    assert np.array_equal(A3, A4) and np.array_equal(b3, b4)
