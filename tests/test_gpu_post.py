"""Parity of the post-differencing calls (sfft_median_combine, sfft_aperture_stats, sfft_cut_stamps,
sfft_multi_template_difference, sfft_resample_*) against
oracle/post_oracle.py, through the C ABI.  Median: bit-exact (it selects values, or averages two).
Aperture fluxes: 1e-12 of sum|D| over the disc (the summation order differs); dropped positions
must agree exactly; sigma to 1e-10 relative."""
import numpy as np
import pytest
import torch

from oracle import post_oracle as po
from paper_2603_08593_b200 import aperture_stats, median_combine

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("n", [1, 2, 3, 4, 5, 6, 7, 8, 9])
@pytest.mark.parametrize("shape", [(37, 53), (64, 128), (1, 1), (3, 333)])
def test_median_combine_bit_exact(n, shape):
    rng = np.random.default_rng(n * 100 + shape[0])
    Ds = [40.0 * rng.standard_normal(shape) for _ in range(n)]
    for D in Ds[:2]:   # ties and repeated values
        D[rng.random(shape) < 0.2] = 1.5
    sc = rng.uniform(0.7, 1.4, n)
    out = median_combine([torch.from_numpy(D).cuda() for D in Ds], sc).cpu().numpy()
    assert np.array_equal(out, po.median_combine(Ds, sc))


@pytest.mark.parametrize("n", [1, 2, 4, 5, 9])
def test_median_combine_nan_propagates(n):
    """Reading M2: a NaN in any template gives a NaN pixel, everything else is untouched (bit-exact)."""
    rng = np.random.default_rng(n)
    Ds = [40.0 * rng.standard_normal((33, 47)) for _ in range(n)]
    Ds[0][5, 6] = np.nan
    Ds[n - 1][32, 46] = np.nan          # odd tail element (33*47 is odd)
    Ds[n // 2][0, 0] = np.nan
    sc = rng.uniform(0.7, 1.4, n)
    out = median_combine([torch.from_numpy(D).cuda() for D in Ds], sc).cpu().numpy()
    ref = po.median_combine(Ds, sc)
    assert np.isnan(ref).sum() == 3
    assert np.array_equal(out, ref, equal_nan=True)


def test_aperture_non_finite_positions_are_dropped():
    D = torch.ones((40, 40), dtype=torch.float64, device="cuda")
    xs = torch.tensor([float("nan"), 20.0, float("inf"), 20.0, 1e300], dtype=torch.float64, device="cuda")
    ys = torch.tensor([20.0, float("-inf"), 20.0, 20.0, 20.0], dtype=torch.float64, device="cuda")
    flux, st = aperture_stats(D, None, xs, ys, 3.0)
    fo, (cnt, mean, sigma) = po.aperture_stats(np.ones((40, 40)), None, xs.cpu().numpy(), ys.cpu().numpy(), 3.0)
    assert np.array_equal(np.isnan(flux.cpu().numpy()), np.isnan(fo)) and cnt == 1
    assert flux[3].item() == 29 and st[0].item() == 1


def test_median_combine_full_ccd_sampled():
    """5 templates at the full CCD size (the launch bench.py times): sampled pixels against the
    definition, and the order-statistic property min <= median <= max everywhere."""
    H, W, n = 2048, 4096, 5
    g = torch.Generator(device="cuda").manual_seed(5)
    Ds = [torch.randn((H, W), dtype=torch.float64, device="cuda", generator=g) * 40 for _ in range(n)]
    sc = [1.0, 0.93, 1.1, 0.8, 1.25]
    out = median_combine(Ds, sc)
    stack = torch.stack([D * s for D, s in zip(Ds, sc)])
    assert bool((out >= stack.min(0).values).all()) and bool((out <= stack.max(0).values).all())
    assert int(((stack < out).sum(0) == 2).sum()) == H * W      # exactly two values below the median (no ties)
    rng = np.random.default_rng(0)
    ys, xs = rng.integers(0, H, 200), rng.integers(0, W, 200)
    host = [D.cpu().numpy() for D in Ds]
    for y, x in zip(ys, xs):
        assert out[y, x].item() == sorted(sc[k] * host[k][y, x] for k in range(n))[2]


@pytest.mark.parametrize("radius", [1.0, 2.7, 4.2, 9.5])
def test_aperture_stats_parity(radius):
    rng = np.random.default_rng(int(radius * 10))
    H, W, n = 300, 420, 1024
    D = 40.0 * rng.standard_normal((H, W)) + 3.0
    mask = (rng.random((H, W)) < 0.002).astype(np.uint8)
    xs, ys = rng.uniform(-2, W + 2, n), rng.uniform(-2, H + 2, n)   # some positions leave the frame
    fo, (cnt, mean, sigma) = po.aperture_stats(D, mask, xs, ys, radius)
    dev = lambda a: torch.from_numpy(a).cuda()
    fg, st = aperture_stats(dev(D), dev(mask), dev(xs), dev(ys), radius)
    fg, st = fg.cpu().numpy(), st.cpu().numpy()
    assert np.array_equal(np.isnan(fg), np.isnan(fo))
    assert 0 < cnt < n
    keep = ~np.isnan(fo)
    scale = 40.0 * 4 * radius * radius + 10
    assert np.max(np.abs(fg[keep] - fo[keep])) <= 1e-12 * scale
    assert st[0] == cnt
    assert abs(st[1] - mean) <= 1e-10 * abs(sigma)
    assert abs(st[2] - sigma) <= 1e-10 * sigma
    # no mask: nothing but the frame edge drops a position
    fg2, st2 = aperture_stats(dev(D), None, dev(xs), dev(ys), radius)
    fo2, (c2, m2, s2) = po.aperture_stats(D, None, xs, ys, radius)
    assert int(st2[0].item()) == c2 and abs(st2[2].item() - s2) <= 1e-10 * s2


def test_aperture_all_dropped_gives_nan_stats():
    D = torch.ones((32, 32), dtype=torch.float64, device="cuda")
    xs = torch.tensor([0.0, 31.0], dtype=torch.float64, device="cuda")
    ys = torch.tensor([0.0, 31.0], dtype=torch.float64, device="cuda")
    flux, st = aperture_stats(D, None, xs, ys, 3.0)
    assert bool(torch.isnan(flux).all()) and st[0].item() == 0 and bool(torch.isnan(st[1:]).all())


@pytest.mark.parametrize("a", [1, 2, 3, 4])
def test_resample_affine_parity(a):
    """Lanczos-a resampling through a rotation + scale + shift: element by element against the oracle
    (1e-13 of the image scale; the weights come from sinpi on the device and math.sin on the host),
    the outside flags exactly."""
    from paper_2603_08593_b200 import resample_affine, resample_mask_affine
    rng = np.random.default_rng(a)
    Hin, Win, Hout, Wout = 70, 90, 64, 80
    img = 40.0 * rng.standard_normal((Hin, Win)) + 100.0
    M = [-1.7, 0.999, 0.012, 2.6, -0.011, 1.002]   # the left columns map outside the frame
    oo, oout = po.resample_affine(img, M, Hout, Wout, a)
    go, gout = resample_affine(torch.from_numpy(img).cuda(), M, Hout, Wout, a)
    assert np.array_equal(gout.cpu().numpy(), oout)
    assert 0 < oout.sum() < oout.size
    assert np.max(np.abs(go.cpu().numpy() - oo)) <= 1e-13 * 300.0
    mask = (rng.random((Hin, Win)) < 0.02).astype(np.uint8)
    om = po.resample_mask_affine(mask, M, Hout, Wout, a, 0.3)
    gm = resample_mask_affine(torch.from_numpy(mask).cuda(), M, Hout, Wout, a, 0.3).cpu().numpy()
    # a value within rounding of the threshold may flip: none does for these inputs
    assert np.array_equal(gm, om) and set(np.unique(gm)) <= {1, 2}


def test_resample_identity_is_bit_exact_on_gpu():
    from paper_2603_08593_b200 import resample_affine
    img = torch.randn((128, 256), dtype=torch.float64, device="cuda")
    out, outside = resample_affine(img, [0, 1, 0, 0, 0, 1], 128, 256, 3)
    inner = outside == 0
    assert bool(inner[2:125, 2:253].all()) and torch.equal(out[inner], img[inner])
    out, outside = resample_affine(img, [5, 1, 0, -2, 0, 1], 128, 256, 3)   # integer shift
    assert torch.equal(out[10:100, 10:200], img[8:98, 15:205])


# ------------------------------------------------------------------- stamps (NEXT-3)
@pytest.mark.parametrize("H,W,size,n", [(40, 56, 7, 40), (64, 64, 63, 9), (33, 47, 4, 25), (16, 16, 1, 10)])
def test_cut_stamps_bit_exact(H, W, size, n):
    """A gather: bit-exact against the oracle, including stamps that hang over every edge, positions
    wholly outside the frame, half-pixel positions and non-finite positions (all-NaN stamps)."""
    from paper_2603_08593_b200 import cut_stamps
    rng = np.random.default_rng(H * 3 + size)
    S, R, D = (rng.standard_normal((H, W)) for _ in range(3))
    xs = rng.uniform(-size, W + size, n)
    ys = rng.uniform(-size, H + size, n)
    xs[:6] = [0.0, W - 1.0, 2.5, -0.5, W + 5.0 * size, 1e300]
    ys[:6] = [0.0, H - 1.0, 3.5, H - 0.5, 1.0, 2.0]
    xs[6], ys[7] = np.nan, np.inf
    ref = po.cut_stamps(S, R, D, xs, ys, size)
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    out = cut_stamps(t(S), t(R), t(D), t(xs), t(ys), size).cpu().numpy()
    assert out.shape == (n, 3, size, size)
    assert np.array_equal(out, ref, equal_nan=True)
    assert np.isnan(ref[6]).all() and np.isnan(ref[7]).all() and not np.isnan(ref[:6]).any()


# ------------------------------------------------------ multi-template mode (NEXT-2)
def _templates(seed, H, W, n):
    rng = np.random.default_rng(seed)
    base = 50.0 * rng.standard_normal((H, W)) + 500.0 * (rng.random((H, W)) > 0.98)
    Rs = [base + 4.0 * rng.standard_normal((H, W)) for _ in range(n)]
    S = 0.7 * np.roll(base, (1, -1), (0, 1)) + 30.0 * rng.standard_normal((H, W)) + 200.0
    mask = (rng.random((H, W)) < 0.03).astype(np.uint8)
    return Rs, S, mask


@pytest.mark.parametrize("H,W,w,DK,DB,n,masked", [(64, 64, 2, 1, 1, 5, True), (1024, 64, 2, 2, 2, 5, True),
                                                   (128, 256, 3, 2, 1, 3, False), (1024, 32, 1, 0, 0, 4, True)])
def test_multi_template_mode_parity_and_reuse(H, W, w, DK, DB, n, masked):
    """sfft_multi_template_difference (the science image's row transform computed once, reused by the
    other templates) against the oracle chain: every D_k and the median at 1e-6 sigma_sky, every c_k
    at 1e-7; and bitwise equal to n separate build/solve/subtract calls plus sfft_median_combine.
    Covers the fused (H = 1024) and the generic column paths."""
    from paper_2603_08593_b200 import SfftPlan, median_combine
    Rs, S, mask = _templates(H + W + n, H, W, n)
    if not masked:
        mask = None
    scales = list(np.linspace(0.9, 1.1, n))
    Dm_o, Ds_o, cs_o = po.multi_template_difference(Rs, S, mask, w, DK, DB, scales, workers=8)
    t = lambda a: None if a is None else torch.from_numpy(np.ascontiguousarray(a)).cuda()
    Rd, Sd, Md = [t(R) for R in Rs], t(S), t(mask)
    sky = 30.0
    with SfftPlan(H, W, w, DK, DB) as plan:
        out, Dk, coeffs, info = plan.multi_template_difference(Rd, Sd, Md, scales)
        torch.cuda.synchronize()
        assert info.cpu().tolist() == [0] * n
        for k in range(n):
            assert np.max(np.abs(coeffs[k].cpu().numpy() - cs_o[k])) <= 1e-7 * np.max(np.abs(cs_o[k]))
            assert np.max(np.abs(Dk[k].cpu().numpy() - Ds_o[k])) <= 1e-6 * sky
        assert np.max(np.abs(out.cpu().numpy() - Dm_o)) <= 1e-6 * sky * max(scales)
        # the reuse changes nothing: separate calls give the same bits
        sep = []
        for k in range(n):
            A, b, c, inf1, D = plan.difference(Rd[k], Sd, Md)
            assert torch.equal(c, coeffs[k]) and torch.equal(D, Dk[k])
            sep.append(D)
        assert torch.equal(median_combine(sep, scales), out)


@pytest.mark.parametrize("H,W,w,DK,DB,n,nplans", [(1024, 64, 2, 2, 2, 5, 3), (64, 64, 2, 1, 1, 5, 2),
                                                   (128, 256, 3, 2, 1, 3, 3), (1024, 32, 1, 0, 0, 2, 3)])
def test_multi_template_mode_over_several_plans(H, W, w, DK, DB, n, nplans):
    """sfft_multi_template_difference_plans (template k on plans[k % nplans], helper plans on their own
    streams, each with the 16-CTA solve grid bench.py uses): every output bitwise equal to the
    single-plan call, twice in a row (the second call finds the plans' scratch used by the first), and
    the chain against the oracle at the parity tolerances.  nplans > n leaves the extra plans idle."""
    from paper_2603_08593_b200 import SfftPlan
    Rs, S, mask = _templates(7 * H + W + n, H, W, n)
    scales = list(np.linspace(1.1, 0.9, n))
    Dm_o, Ds_o, cs_o = po.multi_template_difference(Rs, S, mask, w, DK, DB, scales, workers=8)
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    Rd, Sd, Md = [t(R) for R in Rs], t(S), t(mask)
    sky = 30.0
    plans = [SfftPlan(H, W, w, DK, DB) for _ in range(nplans)]
    try:
        ref = plans[0].multi_template_difference(Rd, Sd, Md, scales)
        for pl in plans:
            pl.set_solve_ctas(16)
        st = torch.cuda.Stream()
        st.wait_stream(torch.cuda.current_stream())
        for rep in range(2):
            with torch.cuda.stream(st):
                got = plans[0].multi_template_difference(Rd, Sd, Md, scales, stream=st, helpers=plans[1:])
                after = got[0] + 1.0          # work enqueued after the call sees the joined result
            st.synchronize()
            for a, b in zip(got, ref):
                assert torch.equal(a, b)
            assert torch.equal(after, ref[0] + 1.0)
        out, Dk, coeffs, info = got
        assert info.cpu().tolist() == [0] * n
        for k in range(n):
            assert np.max(np.abs(coeffs[k].cpu().numpy() - cs_o[k])) <= 1e-7 * np.max(np.abs(cs_o[k]))
            assert np.max(np.abs(Dk[k].cpu().numpy() - Ds_o[k])) <= 1e-6 * sky
        assert np.max(np.abs(out.cpu().numpy() - Dm_o)) <= 1e-6 * sky * max(scales)
        # a helper of another configuration, or the same plan twice, is refused before anything is enqueued
        with SfftPlan(H, W, w, DK, max(DB - 1, 0) if DB else 1) as other:
            with pytest.raises(Exception):
                plans[0].multi_template_difference(Rd, Sd, Md, scales, helpers=[other])
        with pytest.raises(Exception):
            plans[0].multi_template_difference(Rd, Sd, Md, scales, helpers=[plans[0]])
    finally:
        for pl in plans:
            pl.close()


def test_multi_template_mode_rejects_an_artefact_in_one_template():
    from paper_2603_08593_b200 import SfftPlan
    Rs, S, mask = _templates(77, 64, 64, 1)
    R = Rs[0]
    Rbad = R.copy()
    Rbad[20:24, 30:34] += 5000.0
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    with SfftPlan(64, 64, 2, 0, 0) as plan:
        clean, _, _, _ = plan.multi_template_difference([t(R)] * 5, t(S), t(mask), [1.0] * 5)
        mixed, Dk, _, _ = plan.multi_template_difference([t(R), t(R), t(Rbad), t(R), t(R)], t(S), t(mask), [1.0] * 5)
        assert torch.equal(clean, mixed)
        assert float((Dk[2] - clean).abs().max()) > 100.0
