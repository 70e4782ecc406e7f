"""Parity of the CUDA path (through the C ABI) against the CPU oracle, element by element.

Tolerances (BASELINE.json north_star; norms per DESIGN.md reading A5):
  A, b   : max|dA| <= 1e-10 max|A|  and per block (K-K, K-B, B-B, b_K, b_B) <= 1e-12 of the block max
  coeffs : ||c_gpu - c_orc||_inf <= 1e-7 ||c_orc||_inf
  D      : max|dD| <= 1e-6 sigma_sky
"""
import numpy as np
import pytest
import torch

from oracle import sfft_oracle as orc
from paper_2603_08593_b200 import SfftError, SfftPlan, synth

pytestmark = pytest.mark.gpu

TOL_AB = 1e-10
TOL_BLOCK = 1e-12
TOL_C = 1e-7
TOL_D = 1e-6


def dev(x, dtype=None):
    t = torch.from_numpy(np.ascontiguousarray(x))
    if dtype is not None:
        t = t.to(dtype)
    return t.cuda()


def check_system(A, b, Ao, bo, L, TK):
    nK = L * TK
    assert np.max(np.abs(A - Ao)) <= TOL_AB * np.max(np.abs(Ao))
    assert np.max(np.abs(b - bo)) <= TOL_AB * np.max(np.abs(bo))
    blocks = {
        "KK": (A[:nK, :nK], Ao[:nK, :nK]), "KB": (A[:nK, nK:], Ao[:nK, nK:]),
        "BK": (A[nK:, :nK], Ao[nK:, :nK]), "BB": (A[nK:, nK:], Ao[nK:, nK:]),
        "bK": (b[:nK], bo[:nK]), "bB": (b[nK:], bo[nK:]),
    }
    for name, (g, o) in blocks.items():
        scale = max(np.max(np.abs(o)), 1e-300)
        err = np.max(np.abs(g - o))
        assert err <= TOL_BLOCK * scale, (name, err / scale)
    assert np.array_equal(A, A.T)


def run_case(R, S, mask, w, DK, DB, sky_rms, full_D=True):
    H, W = R.shape
    Ao, bo = orc.build_system_fft(R, S, mask, w, DK, DB, workers=8)
    co = orc.solve(Ao, bo)
    with SfftPlan(H, W, w, DK, DB) as plan:
        Rd, Sd = dev(R), dev(S)
        Md = None if mask is None else dev(mask)
        A, b, c, info, D = plan.difference(Rd, Sd, Md)
        torch.cuda.synchronize()
        A, b, c, D = A.cpu().numpy(), b.cpu().numpy(), c.cpu().numpy(), D.cpu().numpy()
        assert int(info.item()) == 0
        L = (2 * w + 1) ** 2
        TK = (DK + 1) * (DK + 2) // 2
        check_system(A, b, Ao, bo, L, TK)
        assert np.max(np.abs(c - co)) <= TOL_C * np.max(np.abs(co))
        # stage-isolated: oracle A, b -> sfft_solve; oracle c -> sfft_subtract
        c2, info2 = plan.solve(dev(Ao), dev(bo))
        assert int(info2.item()) == 0
        assert np.max(np.abs(c2.cpu().numpy() - co)) <= TOL_C * np.max(np.abs(co))
        D2 = plan.subtract(Rd, Sd, dev(co)).cpu().numpy()
    if full_D:
        Do = orc.subtract_rollsum(R, S, co, w, DK, DB)
        assert np.max(np.abs(D2 - Do)) <= TOL_D * sky_rms
        assert np.max(np.abs(D - Do)) <= TOL_D * sky_rms
    else:
        rng = np.random.default_rng(5)
        ys = np.concatenate([rng.integers(0, H, 60), [0, 0, H - 1, H - 1, 3]])
        xs = np.concatenate([rng.integers(0, W, 60), [0, W - 1, 0, W - 1, 2]])
        Dp = orc.subtract_at_pixels(R, S, co, w, DK, DB, ys, xs)
        assert np.max(np.abs(D2[ys, xs] - Dp)) <= TOL_D * sky_rms
        assert np.max(np.abs(D[ys, xs] - Dp)) <= TOL_D * sky_rms
        Df = orc.subtract_fft(R, S, co, w, DK, DB, workers=8)
        assert np.max(np.abs(D2 - Df)) <= TOL_D * sky_rms
        assert np.max(np.abs(D - Df)) <= TOL_D * sky_rms
    return A, b, c, D


def test_tiny_config():
    pr = synth.make_pair("tiny")
    run_case(pr.R, pr.S, pr.mask, pr.cfg.w, pr.cfg.DK, pr.cfg.DB, pr.sky_rms)


def test_small_config():
    pr = synth.make_pair("small", force_saturated=3)
    assert pr.mask[10:-10, 10:-10].any()  # saturated cores are exercised
    run_case(pr.R, pr.S, pr.mask, pr.cfg.w, pr.cfg.DK, pr.cfg.DB, pr.sky_rms)


@pytest.mark.parametrize("H,W,w,DK,DB,masked", [
    (32, 64, 1, 0, 3, True), (128, 32, 2, 3, 0, True), (64, 128, 3, 1, 2, False),
    (512, 64, 0, 2, 1, True), (32, 32, 5, 1, 1, True)])
def test_ragged_shapes_and_degrees(H, W, w, DK, DB, masked):
    rng = np.random.default_rng(H * 7 + W)
    R = 50.0 * rng.standard_normal((H, W)) + 500.0 * (rng.random((H, W)) > 0.98)
    S = 0.7 * np.roll(R, (1 if w else 0, -1 if w else 0), (0, 1)) + 30.0 * rng.standard_normal((H, W)) + 200.0
    mask = (rng.random((H, W)) < 0.05).astype(np.uint8) if masked else None
    run_case(R, S, mask, w, DK, DB, 30.0)


@pytest.mark.parametrize("H,W,w,DK,DB,masked", [
    (16, 16, 3, 1, 1, True), (16, 16, 0, 0, 0, False), (16, 64, 2, 2, 0, True), (128, 16, 1, 0, 2, False),
    (16, 32, 3, 1, 2, True), (2048, 16, 2, 1, 1, True)])
def test_smallest_frame_sizes(H, W, w, DK, DB, masked):
    """H or W = 16, the smallest size include/sfft.h admits (4w+1 <= min(H, W) caps w at 3 there): one
    single-pass transform per row (8 complex points) or column; the last case takes the blocked
    column/cross kernel with 8-point packed rows and a last block of 8 centre rows (fewer than 16 - 2w)."""
    rng = np.random.default_rng(H * 11 + W)
    R = 50.0 * rng.standard_normal((H, W)) + 500.0 * (rng.random((H, W)) > 0.97)
    S = 0.8 * np.roll(R, (1 if w else 0, -1 if w else 0), (0, 1)) + 30.0 * rng.standard_normal((H, W)) + 150.0
    mask = (rng.random((H, W)) < 0.04).astype(np.uint8) if masked else None
    run_case(R, S, mask, w, DK, DB, 30.0)


@pytest.mark.parametrize("H,W,w,DK,DB,masked", [
    (1024, 32, 0, 0, 0, True), (1024, 64, 1, 1, 3, True), (1024, 32, 2, 2, 1, False),
    (2048, 32, 3, 2, 2, True), (1024, 128, 5, 1, 0, True), (4096, 32, 2, 2, 2, True),
    (1024, 64, 4, 3, 1, True),
    # DK = 0 with more blocks per column than ring slots (one task per block), and a short last block
    (2048, 32, 2, 0, 0, True), (4096, 32, 1, 0, 1, False), (2048, 64, 1, 0, 0, True), (2048, 32, 2, 1, 2, True)])
def test_fused_column_cross_path(H, W, w, DK, DB, masked):
    """H in {1024, 2048, 4096}: the fused column-FFT + cross-spectra kernel (every residue-class
    count DR = 2, 4, 8, every instantiated lag range) against the oracle; DK = 3 (> 32 map pairs)
    must fall back to the separate kernels at the same sizes."""
    rng = np.random.default_rng(H + 13 * W + w)
    R = 50.0 * rng.standard_normal((H, W)) + 500.0 * (rng.random((H, W)) > 0.98)
    S = 0.7 * np.roll(R, (1 if w else 0, -1 if w else 0), (0, 1)) + 30.0 * rng.standard_normal((H, W)) + 200.0
    mask = (rng.random((H, W)) < 0.03).astype(np.uint8) if masked else None
    with SfftPlan(H, W, w, DK, DB) as plan:
        assert plan.fused == (DK <= 2)
    run_case(R, S, mask, w, DK, DB, 30.0, full_D=False)


@pytest.mark.parametrize("H,W,w,DK,DB", [
    (32, 64, 6, 1, 1), (32, 32, 7, 0, 0), (64, 64, 6, 2, 2), (64, 128, 8, 1, 0), (128, 64, 10, 1, 2),
    (64, 64, 15, 0, 1), (64, 64, 11, 1, 1), (64, 64, 12, 0, 2), (64, 64, 13, 1, 0), (1024, 64, 6, 2, 1),
    (2048, 32, 7, 1, 1), (64, 256, 9, 3, 0)])
def test_kernel_half_widths_above_five(H, W, w, DK, DB):
    """w = 6 .. 15 (lag half-ranges 12 .. 30): the cross kernel covers the lag range in windows of 25 lags
    (1 window up to half-range 12, 3 above), the lag transform runs its 30-lag instantiation, the sparse
    kernel-background kernel spreads L > 128 shifts over several CTAs and the mixing runs the plain kernel;
    H >= 1024 falls back from the blocked column kernel to the generic column and cross kernels.  The
    exact-objective system is compared too wherever N <= 2047 lets it run."""
    rng = np.random.default_rng(H * 13 + W * 7 + w * 3 + DK)
    R = 50.0 * rng.standard_normal((H, W)) + 500.0 * (rng.random((H, W)) > 0.97)
    S = 0.8 * np.roll(R, (1, -1), (0, 1)) + 30.0 * rng.standard_normal((H, W)) + 150.0
    mask = (rng.random((H, W)) < 0.03).astype(np.uint8)
    run_case(R, S, mask, w, DK, DB, 30.0, full_D=False)
    N = orc.num_coeffs(w, DK, DB)
    with SfftPlan(H, W, w, DK, DB) as plan:
        assert not plan.fused
        if N <= 2047:
            Ax, bx = orc.build_system_exact_fft(R, S, mask, w, DK, DB, workers=8)
            Ae, be = plan.build_system_exact(dev(R), dev(S), dev(mask))
            torch.cuda.synchronize()
            check_system(Ae.cpu().numpy(), be.cpu().numpy(), Ax, bx, (2 * w + 1) ** 2, (DK + 1) * (DK + 2) // 2)
        else:
            with pytest.raises(SfftError) as e:
                plan.build_system_exact(dev(R), dev(S), dev(mask))
            assert e.value.code == 2


@pytest.mark.parametrize("H,W", [(1024, 32), (2048, 32), (4096, 32), (2048, 64), (1024, 16)])
def test_blocked_column_kernel_every_lag_range_and_degree(H, W):
    """sfft_build_system on the blocked column/cross kernel for EVERY kernel half-width 0..5 (the block length
    128 - 4w, the number of blocks per column and the length of the last block all depend on w and H) and
    TK = 1, 3, 6 (the three task tables), plus DK = 3 on the generic kernels, against the oracle."""
    for w in range(0, 6):
        if 4 * w + 1 > min(H, W):
            continue
        for DK, DB in [(0, 0), (1, 2), (2, 1), (0, 3), (3, 0)]:
            rng = np.random.default_rng(H * 13 + W * 7 + w * 3 + DK)
            R = 50.0 * rng.standard_normal((H, W)) + 500.0 * (rng.random((H, W)) > 0.97)
            S = 0.8 * np.roll(R, (1 if w else 0, -1 if w else 0), (0, 1)) + 30.0 * rng.standard_normal((H, W)) + 150.0
            mask = (rng.random((H, W)) < 0.03).astype(np.uint8)
            Ao, bo = orc.build_system_fft(R, S, mask, w, DK, DB, workers=8)
            with SfftPlan(H, W, w, DK, DB) as plan:
                assert plan.fused == (DK <= 2)
                A, b = plan.build_system(dev(R), dev(S), dev(mask))
                torch.cuda.synchronize()
                check_system(A.cpu().numpy(), b.cpu().numpy(), Ao, bo, (2 * w + 1) ** 2, (DK + 1) * (DK + 2) // 2)


def test_mid_config():
    pr = synth.make_pair("mid")
    run_case(pr.R, pr.S, pr.mask, pr.cfg.w, pr.cfg.DK, pr.cfg.DB, pr.sky_rms, full_D=False)


def test_full_config_and_sampled_definition_entries():
    """BASELINE.json configs[3] at full size, in the launch configuration bench.py times; A is
    compared entry by entry with the Fourier-route oracle and, on sampled entries, with direct
    pixel sums of the definition."""
    pr = synth.make_pair("full")
    cfg = pr.cfg
    A, b, c, D = run_case(pr.R, pr.S, pr.mask, cfg.w, cfg.DK, cfg.DB, pr.sky_rms, full_D=False)
    rng = np.random.default_rng(9)
    N = cfg.N
    scale = np.max(np.abs(A))
    for _ in range(12):
        i, j = rng.integers(0, N, 2)
        assert abs(A[i, j] - orc.normal_entry(pr.R, pr.S, pr.mask, cfg.w, cfg.DK, cfg.DB, i, j)) <= TOL_AB * scale
    for i in (0, 60, 725, 731):
        assert abs(b[i] - orc.normal_entry(pr.R, pr.S, pr.mask, cfg.w, cfg.DK, cfg.DB, i)) <= TOL_AB * np.max(np.abs(b))


def test_transposed_ccd_orientation():
    """H=4096, W=2048 (the physical DECam orientation; reading A4)."""
    pr = synth.make_pair("full_t")
    cfg = pr.cfg
    run_case(pr.R, pr.S, pr.mask, cfg.w, cfg.DK, cfg.DB, pr.sky_rms, full_D=False)


def test_exact_recovery_on_gpu():
    """mask=NULL, S = M(R; c0): the CUDA path alone recovers c0 to 1e-9 relative and D = 0."""
    H, W, w, DK, DB = 128, 256, 2, 2, 2
    R, _ = synth.white_noise_pair(H, W, 77)
    rng = np.random.default_rng(1)
    L, TK, TB = 25, 6, 6
    c0 = np.zeros(L * TK + TB)
    c0[:L] = rng.random(L)
    c0[:L] /= c0[:L].sum()
    c0[L:L * TK] = 0.1 * rng.standard_normal(L * (TK - 1))
    c0[L * TK:] = [300.0, 20.0, -10.0, 5.0, 3.0, -4.0]
    S = orc.model_rollsum(R, c0, w, DK, DB)
    with SfftPlan(H, W, w, DK, DB) as plan:
        A, b, c, info, D = plan.difference(dev(R), dev(S), None)
        assert int(info.item()) == 0
        assert np.max(np.abs(c.cpu().numpy() - c0)) <= 1e-9 * np.max(np.abs(c0))
        assert float(D.abs().max()) <= 1e-9 * np.max(np.abs(S))


def test_maximum_size_integer_shift_property():
    """Largest supported frame (4096 x 4096, w = 5, DK = DB = 2, N = 732; fused path with 8 residue
    classes): no oracle at this size, so a property that holds at any size is checked -- with
    mask = NULL and S = roll(R, (v0, u0)) + beta0 the fit is the single delta at (u0, v0) plus the
    constant background, and D vanishes."""
    H = W = 4096
    w, DK, DB = 5, 2, 2
    g = torch.Generator(device="cuda").manual_seed(11)
    R = torch.randn((H, W), dtype=torch.float64, device="cuda", generator=g) * 50.0
    u0, v0, beta0 = -3, 2, 100.0
    S = torch.roll(R, shifts=(v0, u0), dims=(0, 1)) + beta0
    with SfftPlan(H, W, w, DK, DB) as plan:
        assert plan.fused
        A, b, c, info, D = plan.difference(R, S, None)
        assert int(info.item()) == 0
        L = (2 * w + 1) ** 2
        c0 = torch.zeros_like(c)
        c0[(v0 + w) * (2 * w + 1) + (u0 + w)] = 1.0
        c0[L * 6] = beta0
        assert float((c - c0).abs().max()) <= 1e-9 * beta0
        assert float(D.abs().max()) <= 1e-8 * beta0
        assert torch.equal(A, A.T)


def test_not_positive_definite_reports_info():
    H = W = 64
    with SfftPlan(H, W, 1, 0, 0) as plan:
        R = torch.zeros((H, W), dtype=torch.float64, device="cuda")
        S = torch.ones((H, W), dtype=torch.float64, device="cuda")
        A, b = plan.build_system(R, S, None)
        c, info = plan.solve(A, b)
        assert int(info.item()) == 1


def test_degenerate_all_masked_and_plan_reuse():
    pr = synth.make_pair("tiny")
    cfg = pr.cfg
    with SfftPlan(cfg.H, cfg.W, cfg.w, cfg.DK, cfg.DB) as plan:
        allm = torch.ones((cfg.H, cfg.W), dtype=torch.uint8, device="cuda")
        A, b = plan.build_system(dev(pr.R), dev(pr.S), allm)
        assert float(A.abs().max()) == 0.0 and float(b.abs().max()) == 0.0
        # the same plan gives the same answer when reused (scratch holds no state)
        A1, b1 = plan.build_system(dev(pr.R), dev(pr.S), dev(pr.mask))
        A2, b2 = plan.build_system(dev(pr.R), dev(pr.S), dev(pr.mask))
        assert torch.equal(A1, A2) and torch.equal(b1, b2)
        assert plan.last_launch_count(0) > 0


@pytest.mark.parametrize("cfg", [(2048, 4096, 5, 2, 2), (256, 256, 3, 1, 1), (32, 32, 0, 0, 0)])
def test_solve_is_bitwise_independent_of_the_cta_cap(cfg):
    """include/sfft.h, sfft_plan_set_solve_ctas: "Results are bitwise independent of the setting" -- grids of
    1, 3, 16, 50 CTAs and the default (one per SM) on N = 732, 150 and 2, against the oracle's solve too."""
    with SfftPlan(*cfg) as plan:
        N = plan.N
        rng = np.random.default_rng(N)
        G = rng.standard_normal((2 * N + 20, N))
        A = G.T @ G + 1e-3 * np.eye(N)
        b = rng.standard_normal(N)
        co = orc.solve(A, b)
        Ad, bd = dev(A), dev(b)
        ref = None
        for cap in (0, 1, 3, 16, 50):
            plan.set_solve_ctas(cap)
            c, info = plan.solve(Ad, bd)
            torch.cuda.synchronize()
            assert int(info.item()) == 0
            if ref is None:
                ref = c.clone()
                assert np.max(np.abs(ref.cpu().numpy() - co)) <= TOL_C * np.max(np.abs(co))
            else:
                assert torch.equal(c, ref), cap


def test_non_default_stream():
    pr = synth.make_pair("tiny")
    cfg = pr.cfg
    st = torch.cuda.Stream()
    with SfftPlan(cfg.H, cfg.W, cfg.w, cfg.DK, cfg.DB) as plan:
        Rd, Sd, Md = dev(pr.R), dev(pr.S), dev(pr.mask)
        torch.cuda.synchronize()
        with torch.cuda.stream(st):
            A, b, c, info, D = plan.difference(Rd, Sd, Md, stream=st)
        st.synchronize()
        A0, b0, c0, info0, D0 = plan.difference(Rd, Sd, Md)
        torch.cuda.synchronize()
        assert torch.equal(D, D0) and torch.equal(c, c0)


def test_subtract_prepare_is_bitwise_neutral_and_safe():
    """sfft_subtract_prepare only moves work: D is bitwise the same with and without it; a prepare for
    another R, or one followed by a new build_system, is discarded."""
    pr = synth.make_pair("small")
    cfg = pr.cfg
    with SfftPlan(cfg.H, cfg.W, cfg.w, cfg.DK, cfg.DB) as plan:
        R, S, M = dev(pr.R), dev(pr.S), dev(pr.mask)
        A, b = plan.build_system(R, S, M)
        c, info = plan.solve(A, b)
        D0 = plan.subtract(R, S, c).clone()
        # prepared for the same R
        plan.subtract_prepare(R)
        c1, _ = plan.solve(A, b)
        assert torch.equal(plan.subtract(R, S, c1), D0)
        # prepared for ANOTHER image: must not be used
        R2 = (R * 1.5).contiguous()
        plan.subtract_prepare(R2)
        assert torch.equal(plan.subtract(R, S, c), D0)
        # prepared, then the scratch is reused by a build: must not be used either
        plan.subtract_prepare(R)
        plan.build_system(R, S, M)
        assert torch.equal(plan.subtract(R, S, c), D0)
        # a prepare is consumed by one subtract only
        plan.subtract_prepare(R)
        assert torch.equal(plan.subtract(R, S, c), D0)
        assert torch.equal(plan.subtract(R, S, c), D0)
        torch.cuda.synchronize()


@pytest.mark.parametrize("H,W,w,DK,DB,border", [(64, 64, 2, 0, 0, 2), (128, 64, 2, 1, 1, 0), (64, 256, 3, 2, 2, 3),
                                                (1024, 64, 1, 1, 2, 4), (32, 32, 5, 1, 1, 0)])
def test_exact_objective_parity(H, W, w, DK, DB, border):
    """sfft_build_system_exact (literal objective: masked pixels dropped, images unmasked) against the
    oracle's Fourier-route system minus the masked pixels' rank-one terms; several tiles and slices of
    the rank-K update, ragged tile edges (N + 1 not a multiple of 128), fused and generic plans."""
    rng = np.random.default_rng(H + W + w)
    R = 50.0 * rng.standard_normal((H, W)) + 500.0 * (rng.random((H, W)) > 0.98)
    S = 0.7 * np.roll(R, (1, -1), (0, 1)) + 30.0 * rng.standard_normal((H, W)) + 200.0
    mask = (rng.random((H, W)) < 0.05).astype(np.uint8)
    if border:
        mask[:border] = 1; mask[-border:] = 1; mask[:, :border] = 1; mask[:, -border:] = 1
    Ao, bo = orc.build_system_exact_fft(R, S, mask, w, DK, DB, workers=8)
    with SfftPlan(H, W, w, DK, DB) as plan:
        A, b = plan.build_system_exact(dev(R), dev(S), dev(mask))
        A2, b2 = plan.build_system_exact(dev(R), dev(S), dev(mask))
        assert torch.equal(A, A2) and torch.equal(b, b2)          # reproducible
        A, b = A.cpu().numpy(), b.cpu().numpy()
        L = (2 * w + 1) ** 2
        TK = (DK + 1) * (DK + 2) // 2
        check_system(A, b, Ao, bo, L, TK)
        # mask = None: identical to the ordinary build
        A0, b0 = plan.build_system_exact(dev(R), dev(S), None)
        A1, b1 = plan.build_system(dev(R), dev(S), None)
        assert torch.equal(A0, A1) and torch.equal(b0, b1)


@pytest.mark.parametrize("H,W,w,DK,DB,kind", [
    (128, 128, 2, 1, 1, "frame+lines"), (64, 256, 3, 2, 2, "frame+lines"), (256, 64, 1, 2, 0, "many_rows"),
    (128, 64, 5, 1, 1, "scattered_rows"), (64, 64, 0, 2, 2, "frame+lines"), (128, 128, 2, 0, 3, "cols_only")])
def test_exact_objective_structured_masks(H, W, w, DK, DB, kind):
    """The structured part of sfft_build_system_exact (fully masked rows / columns through strip
    correlations, corners added back, the rest through the pixel list) against the oracle: frames with
    extra full lines in the interior and isolated pixels; more full rows than the strip path accepts
    (the surplus stays in the pixel list); full rows so far apart that the source-line cap is hit;
    w = 0; columns only."""
    rng = np.random.default_rng(7 * H + W + w)
    R = 50.0 * rng.standard_normal((H, W)) + 500.0 * (rng.random((H, W)) > 0.98)
    S = 0.7 * np.roll(R, (1 if w else 0, -1 if w else 0), (0, 1)) + 30.0 * rng.standard_normal((H, W)) + 200.0
    mask = (rng.random((H, W)) < 0.02).astype(np.uint8)
    if kind == "frame+lines":
        mask[:3] = 1; mask[-2:] = 1; mask[:, :2] = 1; mask[:, -3:] = 1
        mask[H // 2] = 1; mask[:, W // 3] = 1; mask[:, W // 3 + 1] = 1
    elif kind == "many_rows":
        mask[10:50] = 1                      # 40 full rows: 32 take the strip path
        mask[:, 5] = 1
    elif kind == "scattered_rows":
        mask[::16] = 1                       # 8 isolated full rows, 11 source rows each: the 64-line cap is hit
    elif kind == "cols_only":
        mask[:, 7:11] = 1; mask[:, -1] = 1
    Ao, bo = orc.build_system_exact_fft(R, S, mask, w, DK, DB, workers=8)
    with SfftPlan(H, W, w, DK, DB) as plan:
        A, b = plan.build_system_exact(dev(R), dev(S), dev(mask))
        A2, b2 = plan.build_system_exact(dev(R), dev(S), dev(mask))
        assert torch.equal(A, A2) and torch.equal(b, b2)          # reproducible
        L = (2 * w + 1) ** 2
        TK = (DK + 1) * (DK + 2) // 2
        check_system(A.cpu().numpy(), b.cpu().numpy(), Ao, bo, L, TK)


def test_exact_objective_recovers_kernel_under_mask_on_gpu():
    """S = M(R; c0) with a border + random mask: the exact objective returns c0 to 1e-9 and D = 0 on
    the GPU path alone; the input-masking system does not (reading A2')."""
    H, W, w, DK, DB = 128, 256, 2, 2, 2
    R, _ = synth.white_noise_pair(H, W, 78)
    rng = np.random.default_rng(2)
    L, TK = 25, 6
    c0 = np.zeros(L * TK + 6)
    c0[:L] = rng.random(L)
    c0[:L] /= c0[:L].sum()
    c0[L:L * TK] = 0.1 * rng.standard_normal(L * (TK - 1))
    c0[L * TK:] = [300.0, 20.0, -10.0, 5.0, 3.0, -4.0]
    S = orc.model_rollsum(R, c0, w, DK, DB)
    mask = (rng.random((H, W)) < 0.06).astype(np.uint8)
    mask[:4] = 1; mask[-4:] = 1; mask[:, :4] = 1; mask[:, -4:] = 1
    with SfftPlan(H, W, w, DK, DB) as plan:
        A, b = plan.build_system_exact(dev(R), dev(S), dev(mask))
        c, info = plan.solve(A, b)
        assert int(info.item()) == 0
        assert np.max(np.abs(c.cpu().numpy() - c0)) <= 1e-9 * np.max(np.abs(c0))
        D = plan.subtract(dev(R), dev(S), c)
        assert float(D.abs().max()) <= 1e-9 * np.max(np.abs(S))
        A2, b2 = plan.build_system(dev(R), dev(S), dev(mask))
        c2, _ = plan.solve(A2, b2)
        assert np.max(np.abs(c2.cpu().numpy() - c0)) > 1e-5 * np.max(np.abs(c0))


def test_exact_objective_full_config_sampled():
    """Full CCD (2048 x 4096, N = 732, ~74 k masked border pixels): sampled entries of A_ex, b_ex
    against direct sums over the unmasked pixels; symmetry; the update is a small correction of the
    unmasked system."""
    pr = synth.make_pair("full")
    cfg = pr.cfg
    with SfftPlan(cfg.H, cfg.W, cfg.w, cfg.DK, cfg.DB) as plan:
        Rd, Sd, Md = dev(pr.R), dev(pr.S), dev(pr.mask)
        A, b = plan.build_system_exact(Rd, Sd, Md)
        c, info = plan.solve(A, b)
        assert int(info.item()) == 0
        A, b = A.cpu().numpy(), b.cpu().numpy()
    assert np.array_equal(A, A.T)
    rng = np.random.default_rng(3)
    N = cfg.N
    scale = np.max(np.abs(A))
    pairs = [tuple(rng.integers(0, N, 2)) for _ in range(8)] + [(N - 1, N - 1), (N - 3, 17), (0, 0)]
    for i, j in pairs:
        assert abs(A[i, j] - orc.exact_entry(pr.R, pr.S, pr.mask, cfg.w, cfg.DK, cfg.DB, int(i), int(j))) <= TOL_AB * scale
    for i in (0, 61, 725, 731):
        assert abs(b[i] - orc.exact_entry(pr.R, pr.S, pr.mask, cfg.w, cfg.DK, cfg.DB, i)) <= TOL_AB * np.max(np.abs(b))


def test_exposure_configuration_three_plans_in_flight():
    """The launch configuration bench.py's exposure and end-to-end legs time (BASELINE.json configs[4];
    PAPER.md:324, a GPU works through a queue of CCDs): 3 plans on 3 streams in flight at once,
    sfft_plan_set_solve_ctas(16), sfft_subtract_prepare before the solve, exposure-recipe pairs (seed 2000+k) at the
    extremes of the recipe (sky 800 / FWHM 6 and sky 3000 / FWHM 3.5) plus one mid draw.  A, b, c, D of
    the two extreme pairs against the oracle at the A5 tolerances, and every pair bitwise equal to the
    same pair run alone on one plan with the default solve grid (sfft.h: "Results are bitwise
    independent of the setting")."""
    prs = [synth.make_pair("full", seed=2000, sky0=800.0, fwhm_s=6.0),
           synth.make_pair("full", seed=2001, sky0=3000.0, fwhm_s=3.5),
           synth.make_exposure_pair(2)]
    cfg = prs[0].cfg
    N = cfg.N
    devp = [(dev(p.R), dev(p.S), dev(p.mask)) for p in prs]
    streams = [torch.cuda.Stream() for _ in prs]
    plans = [SfftPlan(cfg.H, cfg.W, cfg.w, cfg.DK, cfg.DB) for _ in prs]
    outs = []
    try:
        for pl in plans:
            pl.set_solve_ctas(16)
        torch.cuda.synchronize()
        res = [None] * len(prs)
        for rep in range(2):                      # second round: every plan's scratch has been used once
            for k, (pl, st) in enumerate(zip(plans, streams)):
                R, S, M = devp[k]
                with torch.cuda.stream(st):
                    A, b = pl.build_system(R, S, M, stream=st)
                    pl.subtract_prepare(R, stream=st)
                    c, info = pl.solve(A, b, stream=st)
                    D = pl.subtract(R, S, c, stream=st)
                res[k] = (A, b, c, info, D)
        torch.cuda.synchronize()
        # the same pairs alone, one plan, default grid, with the prepare hint (the single-stream path)
        with SfftPlan(cfg.H, cfg.W, cfg.w, cfg.DK, cfg.DB) as solo:
            for k in range(len(prs)):
                R, S, M = devp[k]
                A0, b0, c0, info0, D0 = solo.difference(R, S, M)
                torch.cuda.synchronize()
                A, b, c, info, D = res[k]
                assert int(info.item()) == 0 and int(info0.item()) == 0
                assert torch.equal(A, A0) and torch.equal(b, b0), k
                assert torch.equal(c, c0), k
                assert torch.equal(D, D0), k
        outs = [tuple(t.cpu().numpy() for t in (r[0], r[1], r[2], r[4])) for r in res[:2]]
    finally:
        for pl in plans:
            pl.close()
    L, TK = cfg.L, (cfg.DK + 1) * (cfg.DK + 2) // 2
    for k, (A, b, c, D) in enumerate(outs):
        pr = prs[k]
        Ao, bo = orc.build_system_fft(pr.R, pr.S, pr.mask, cfg.w, cfg.DK, cfg.DB, workers=8)
        co = orc.solve(Ao, bo)
        check_system(A, b, Ao, bo, L, TK)
        assert np.max(np.abs(c - co)) <= TOL_C * np.max(np.abs(co))
        Df = orc.subtract_fft(pr.R, pr.S, co, cfg.w, cfg.DK, cfg.DB, workers=8)
        assert np.max(np.abs(D - Df)) <= TOL_D * pr.sky_rms
        rng = np.random.default_rng(50 + k)
        ys, xs = rng.integers(0, cfg.H, 20), rng.integers(0, cfg.W, 20)
        Dp = orc.subtract_at_pixels(pr.R, pr.S, co, cfg.w, cfg.DK, cfg.DB, ys, xs)
        assert np.max(np.abs(D[ys, xs] - Dp)) <= TOL_D * pr.sky_rms


def test_difference_host_end_to_end_call():
    """SfftPlan.difference_host (pinned host buffers in, D and coefficients out -- the call bench.py's
    e2e leg times) on a non-default stream equals the device-resident path bitwise."""
    pr = synth.make_pair("small", force_saturated=3)
    cfg = pr.cfg
    hR, hS, hM = (torch.from_numpy(x).pin_memory() for x in (pr.R, pr.S, pr.mask))
    st = torch.cuda.Stream()
    with SfftPlan(cfg.H, cfg.W, cfg.w, cfg.DK, cfg.DB) as plan:
        Dh, ch, ih = plan.difference_host(hR, hS, hM, stream=st)
        assert int(ih.item()) == 0 and not Dh.is_cuda and not ch.is_cuda
        A, b, c, info, D = plan.difference(dev(pr.R), dev(pr.S), dev(pr.mask))
        torch.cuda.synchronize()
        assert torch.equal(Dh, D.cpu()) and torch.equal(ch, c.cpu())
