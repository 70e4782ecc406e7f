"""CPU ORACLE for SFFT image differencing -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference`
legs may import this module.  It shares no code with the CUDA path (paper_2603_08593_b200/csrc)
and does not import the package.  Plain numpy/scipy in float64, written from the definition.

What it computes (§1: "formulates the image subtraction problem in the Fourier
domain and accounts for spatial variations in the point-spread function ... convolution kernel
is modeled with a delta-function basis"; §2.3.2: used once per science image).
The paper gives no equations; BASELINE.json `north_star` fixes the problem and SURVEY.md §8.0 /
§8(c) fix the conventions (readings A1..A14, restated in DESIGN.md):

    D = S - ( R (x) K(x,y) + B(x,y) ),  circular convolution,
    K: (2w+1)^2 delta basis, coefficients = degree-DK polynomials of the SOURCE pixel (A1),
    B: degree-DB polynomial,  coefficients minimise sum D^2 via the normal equations.

    xi(x)  = (2x+1-W)/W,  eta(y) = (2y+1-H)/H                                  (A3)
    monomials P_t = xi^p eta^q ordered  for d in 0..D: for q in 0..d: p=d-q    (A4)
    shifts s <-> (u,v), s=(v+w)(2w+1)+(u+w), u along x, v along y              (A4)
    m = 1 where mask==0 (or mask is None) else 0                               (A12)
    R~_t = m P_t R,  S~ = m S,  Psi_t' = m P_t'                                (A2: input masking)
    G[(y,x),(t,s)] = R~_t[(y-v) mod H, (x-u) mod W];  G[(y,x), L*T_K+t'] = Psi_t'[y,x]
    A = G^T G,  b = G^T S~,  c = A^-1 b  (Cholesky, no regularisation; A8, A9)
    c[t*L+s] = a_{s,t},  c[L*T_K+t'] = beta_t'
    D = S - sum_{s,t} a_{s,t} roll(P_t R,(v,u)) - sum_t' beta_t' P_t'   (UNMASKED R, S)

Pins (tests/test_oracle_pins.py, all `-m "not gpu"`): brute-force G^T G vs the FFT route;
symmetry/PSD/block-Toeplitz invariants; B-B block closed forms by exact rational arithmetic;
scipy.signal.correlate2d on bordered images; identity / integer-shift / exact-recovery of a
known kernel+background; lstsq cross-check; roll-sum D vs Fourier-route D.  No function here is
"parity unpinned".
"""
from __future__ import annotations

import numpy as np
import scipy.fft
import scipy.linalg

# --------------------------------------------------------------------------- conventions


def monomials(D):
    """Exponent pairs (p,q) of xi^p eta^q, ordered by total degree then q."""
    return [(d - q, q) for d in range(D + 1) for q in range(d + 1)]


def shifts(w):
    """Shift list [(u,v)] in index order s=(v+w)(2w+1)+(u+w)."""
    return [(u, v) for v in range(-w, w + 1) for u in range(-w, w + 1)]


def num_coeffs(w, DK, DB):
    return (2 * w + 1) ** 2 * (DK + 1) * (DK + 2) // 2 + (DB + 1) * (DB + 2) // 2


def coords(H, W, dtype=np.float64):
    """Normalised pixel coordinates xi(x), eta(y) in (-1,1) (A3)."""
    xi = (2 * np.arange(W, dtype=dtype) + 1 - W) / dtype(W)
    eta = (2 * np.arange(H, dtype=dtype) + 1 - H) / dtype(H)
    return xi, eta


def _poly_images(H, W, D, dtype=np.float64):
    xi, eta = coords(H, W, dtype)
    return [np.multiply.outer(eta ** q, xi ** p) for (p, q) in monomials(D)]


def _good(mask, shape, dtype=np.float64):
    if mask is None:
        return np.ones(shape, dtype=dtype)
    return (np.asarray(mask) == 0).astype(dtype)


# --------------------------------------------------------------------------- O1: definition


def design_matrix(R, S, mask, w, DK, DB):
    """G (P x N) and the masked target S~ (P), literally as defined."""
    H, W = R.shape
    m = _good(mask, R.shape)
    cols = []
    for Pt in _poly_images(H, W, DK):
        Rt = m * Pt * R
        for (u, v) in shifts(w):
            cols.append(np.roll(Rt, shift=(v, u), axis=(0, 1)).ravel())
    for Pt in _poly_images(H, W, DB):
        cols.append((m * Pt).ravel())
    return np.stack(cols, axis=1), (m * S).ravel()


def build_system_bruteforce(R, S, mask, w, DK, DB):
    """O1: A = G^T G, b = G^T S~ with G formed explicitly (tiny/small sizes)."""
    G, St = design_matrix(R, S, mask, w, DK, DB)
    return G.T @ G, G.T @ St


def normal_entry(R, S, mask, w, DK, DB, i, j=None):
    """One entry A[i,j] (or b[i] when j is None) by a direct pixel sum of two columns of G.
    Lets the full-size CUDA result be checked on sampled entries without forming G."""
    H, W = R.shape
    m = _good(mask, R.shape)
    L = (2 * w + 1) ** 2
    TK = (DK + 1) * (DK + 2) // 2
    xi, eta = coords(H, W)

    def column(idx):
        if idx < L * TK:
            t, s = divmod(idx, L)
            p, q = monomials(DK)[t]
            u, v = shifts(w)[s]
            return np.roll(m * np.multiply.outer(eta ** q, xi ** p) * R, shift=(v, u), axis=(0, 1))
        p, q = monomials(DB)[idx - L * TK]
        return m * np.multiply.outer(eta ** q, xi ** p)

    gi = column(i)
    gj = (m * S) if j is None else column(j)
    return float(np.sum(gi * gj))


# --------------------------------------------------------------------------- O2: Fourier route


def build_system_fft(R, S, mask, w, DK, DB, workers=1, dtype=np.float64):
    """O2: A, b from cross-correlation maps read at the shift differences (north_star (3),(4)).

        A[t L+s, t' L+s'] = C_{t,t'}[(u-u', v-v')]      (K-K block; t>t' by symmetry)
        b[t L+s]          = C_{t,S}[(u,v)]
        A[t L+s, L T_K+t'] = C_{t,Psi_t'}[(u,v)]        (K-B block and its transpose)
        A[B,B], b_B        = direct pixel sums of Psi_t Psi_t', Psi_t S~

    dtype=np.longdouble gives the ~1e-19 accuracy referee O5 (scipy.fft supports long double).
    """
    R = np.asarray(R, dtype=dtype)
    S = np.asarray(S, dtype=dtype)
    H, W = R.shape
    m = _good(mask, R.shape, dtype)
    L = (2 * w + 1) ** 2
    sh = shifts(w)
    polyK = _poly_images(H, W, DK, dtype)
    polyB = _poly_images(H, W, DB, dtype)
    TK, TB = len(polyK), len(polyB)
    N = L * TK + TB
    A = np.zeros((N, N), dtype=dtype)
    b = np.zeros(N, dtype=dtype)

    Rt = [m * Pt * R for Pt in polyK]
    St = m * S
    Psi = [m * Pt for Pt in polyB]
    FR = [scipy.fft.rfft2(x, workers=workers) for x in Rt]
    FS = scipy.fft.rfft2(St, workers=workers)
    FP = [scipy.fft.rfft2(x, workers=workers) for x in Psi]

    def corr(Fa, Fb):
        return scipy.fft.irfft2(np.conj(Fa) * Fb, s=(H, W), workers=workers)

    for t in range(TK):
        for t2 in range(t, TK):
            C = corr(FR[t], FR[t2])
            for s, (u, v) in enumerate(sh):
                for s2, (u2, v2) in enumerate(sh):
                    val = C[(v - v2) % H, (u - u2) % W]
                    A[t * L + s, t2 * L + s2] = val
                    A[t2 * L + s2, t * L + s] = val
        C = corr(FR[t], FS)
        for s, (u, v) in enumerate(sh):
            b[t * L + s] = C[v % H, u % W]
        for t2 in range(TB):
            C = corr(FR[t], FP[t2])
            for s, (u, v) in enumerate(sh):
                val = C[v % H, u % W]
                A[t * L + s, L * TK + t2] = val
                A[L * TK + t2, t * L + s] = val
    for t in range(TB):
        b[L * TK + t] = np.sum(Psi[t] * St)
        for t2 in range(TB):
            A[L * TK + t, L * TK + t2] = np.sum(Psi[t] * Psi[t2])
    return A, b


# --------------------------------------------------------------------------- O3: solve


def solve(A, b):
    """O3: c = A^-1 b by Cholesky (A symmetric positive definite; A9).  Raises LinAlgError
    if a leading minor is not positive (the CUDA path reports that through `info`)."""
    cf = scipy.linalg.cho_factor(np.asarray(A, dtype=np.float64), lower=True)
    return scipy.linalg.cho_solve(cf, np.asarray(b, dtype=np.float64))


# --------------------------------------------------------------------------- O4: difference image


def model_rollsum(R, c, w, DK, DB):
    """M = sum_{t,s} a_{s,t} roll(P_t R,(v,u)) + sum_t' beta_t' P_t'  (unmasked R; A1, A6, A7)."""
    H, W = R.shape
    L = (2 * w + 1) ** 2
    polyK = _poly_images(H, W, DK)
    polyB = _poly_images(H, W, DB)
    M = np.zeros((H, W))
    for t, Pt in enumerate(polyK):
        Q = Pt * R
        for s, (u, v) in enumerate(shifts(w)):
            a = c[t * L + s]
            if a != 0.0:
                M += a * np.roll(Q, shift=(v, u), axis=(0, 1))
    for t, Pt in enumerate(polyB):
        M += c[L * len(polyK) + t] * Pt
    return M


def subtract_rollsum(R, S, c, w, DK, DB):
    """O4: D = S - M, by the explicit roll-sum definition."""
    return S - model_rollsum(R, c, w, DK, DB)


def subtract_fft(R, S, c, w, DK, DB, workers=1):
    """O4 (Fourier route, north_star (6)): M = irfft2( sum_t K^_t * rfft2(P_t R) ) + B with
    K^_t(k) = sum_s a_{s,t} exp(-2 pi i (kx u/W + ky v/H)).  Pinned to subtract_rollsum."""
    H, W = R.shape
    L = (2 * w + 1) ** 2
    polyK = _poly_images(H, W, DK)
    polyB = _poly_images(H, W, DB)
    kx = np.arange(W // 2 + 1)
    ky = np.arange(H)
    acc = np.zeros((H, W // 2 + 1), dtype=np.complex128)
    for t, Pt in enumerate(polyK):
        Khat = np.zeros((H, W // 2 + 1), dtype=np.complex128)
        for s, (u, v) in enumerate(shifts(w)):
            a = c[t * L + s]
            Khat += a * np.multiply.outer(np.exp(-2j * np.pi * ky * v / H),
                                          np.exp(-2j * np.pi * kx * u / W))
        acc += Khat * scipy.fft.rfft2(Pt * R, workers=workers)
    M = scipy.fft.irfft2(acc, s=(H, W), workers=workers)
    for t, Pt in enumerate(polyB):
        M += c[L * len(polyK) + t] * Pt
    return S - M


def subtract_at_pixels(R, S, c, w, DK, DB, ys, xs):
    """D at selected pixels straight from the definition (one pixel at a time; any image size)."""
    H, W = R.shape
    L = (2 * w + 1) ** 2
    monoK, monoB = monomials(DK), monomials(DB)
    xi, eta = coords(H, W)
    out = np.empty(len(ys))
    sh = shifts(w)
    for i, (y, x) in enumerate(zip(ys, xs)):
        mod = 0.0
        for t, (p, q) in enumerate(monoK):
            for s, (u, v) in enumerate(sh):
                yy, xx = (y - v) % H, (x - u) % W
                mod += c[t * L + s] * (xi[xx] ** p) * (eta[yy] ** q) * R[yy, xx]
        for t, (p, q) in enumerate(monoB):
            mod += c[L * len(monoK) + t] * (xi[x] ** p) * (eta[y] ** q)
        out[i] = S[y, x] - mod
    return out


# --------------------------------------------------------------------------- whole path


def sfft_difference(R, S, mask, w, DK, DB, workers=1, fourier_subtract=True):
    """The whole hot path on the CPU: build (O2) -> solve (O3) -> subtract (O4)."""
    A, b = build_system_fft(R, S, mask, w, DK, DB, workers=workers)
    c = solve(A, b)
    if fourier_subtract:
        D = subtract_fft(R, S, c, w, DK, DB, workers=workers)
    else:
        D = subtract_rollsum(R, S, c, w, DK, DB)
    return A, b, c, D


# --------------------------------------------------------------------------- exact objective (NEXT-1)
# BASELINE.json north_star: "the coefficients minimise sum D^2 over unmasked pixels".  Reading A2
# (input masking) is what the Fourier formulation needs; the LITERAL objective keeps R and S as they
# are and drops the masked pixels from the sum:
#     A_ex = sum_{x unmasked} g(x) g(x)^T,   b_ex = sum_{x unmasked} g(x) S(x),
#     g(x) = row x of the design matrix built from the UNMASKED R (and the unmasked P_t').
# Equivalently A_ex = A(mask=None) - sum_{x masked} g(x) g(x)^T.  With it a known kernel is
# recovered exactly under any mask (pinned in tests/test_oracle_pins.py).


def build_system_exact_bruteforce(R, S, mask, w, DK, DB):
    """A_ex, b_ex from the explicit design matrix of the unmasked images, masked rows dropped."""
    G, St = design_matrix(R, S, None, w, DK, DB)
    if mask is None:
        return G.T @ G, G.T @ St
    keep = (np.asarray(mask).ravel() == 0)
    Gk = G[keep]
    return Gk.T @ Gk, Gk.T @ St[keep]


def design_rows(R, mask_pixels, w, DK, DB):
    """Rows g(x) of the unmasked design matrix for the listed pixels [(y, x), ...], by explicit
    index arithmetic (no G of the whole image): used at sizes where G does not fit."""
    H, W = R.shape
    xi, eta = coords(H, W)
    out = np.zeros((len(mask_pixels), num_coeffs(w, DK, DB)))
    sh = shifts(w)
    L = len(sh)
    for r, (y, x) in enumerate(mask_pixels):
        for t, (p, q) in enumerate(monomials(DK)):
            for s, (u, v) in enumerate(sh):
                ys, xs = (y - v) % H, (x - u) % W
                out[r, t * L + s] = xi[xs] ** p * eta[ys] ** q * R[ys, xs]
        for t2, (p, q) in enumerate(monomials(DB)):
            out[r, L * len(monomials(DK)) + t2] = xi[x] ** p * eta[y] ** q
    return out


def build_system_exact_fft(R, S, mask, w, DK, DB, workers=1):
    """A_ex, b_ex as the unmasked Fourier-route system minus the masked pixels' rank-one terms."""
    A, b = build_system_fft(R, S, None, w, DK, DB, workers=workers)
    if mask is None:
        return A, b
    ys, xs = np.nonzero(np.asarray(mask))
    pix = list(zip(ys.tolist(), xs.tolist()))
    A = A.copy()
    b = b.copy()
    for i0 in range(0, len(pix), 4096):   # chunks keep the row block small
        Gm = design_rows(R, pix[i0:i0 + 4096], w, DK, DB)
        Sm = np.array([S[y, x] for (y, x) in pix[i0:i0 + 4096]])
        A -= Gm.T @ Gm
        b -= Gm.T @ Sm
    return A, b


def exact_entry(R, S, mask, w, DK, DB, i, j=None):
    """One entry of A_ex (or of b_ex when j is None) by a direct sum over the unmasked pixels of
    two columns of the UNMASKED design matrix (full-size sampled checks without forming G)."""
    keep = _good(mask, R.shape)
    if j is None:
        G_i = normal_entry_column(R, w, DK, DB, i)
        return float(np.sum(keep * G_i * S))
    return float(np.sum(keep * normal_entry_column(R, w, DK, DB, i) * normal_entry_column(R, w, DK, DB, j)))


def normal_entry_column(R, w, DK, DB, idx):
    """Column idx of the design matrix of the unmasked images, as an H x W image."""
    H, W = R.shape
    L = (2 * w + 1) ** 2
    TK = (DK + 1) * (DK + 2) // 2
    xi, eta = coords(H, W)
    if idx < L * TK:
        t, s = divmod(idx, L)
        p, q = monomials(DK)[t]
        u, v = shifts(w)[s]
        return np.roll(np.multiply.outer(eta ** q, xi ** p) * R, shift=(v, u), axis=(0, 1))
    p, q = monomials(DB)[idx - L * TK]
    return np.multiply.outer(eta ** q, xi ** p)
