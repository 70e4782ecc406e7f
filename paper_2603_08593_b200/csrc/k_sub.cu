// sfft_subtract: application of the fitted spatially varying kernel in the row-Fourier domain
// (north_star subsystem (6)).
//
// The delta-basis model  M(x,y) = sum_t sum_{u,v} a[(u,v),t] (P_t R)(x-u, y-v)  is separable in the
// sense that the x-shift is a phase in the row spectrum and the y-shift a row offset.  With
// G_p = rfft_x(xi^p R) (DK+1 row transforms, no column transforms at all) and
//   E_t[v][kx] = sum_u a[(u,v),t] e^{-2 pi i kx u/W},
//   Mhat[y][kx] = sum_v sum_{t=(p,q)} E_t[v][kx] eta(y-v)^q G_p[(y-v) mod H][kx],
// M = irfft_x(Mhat); k_row_inv_sub (k_rows.cu) finishes with D = S - M - B.  Column 0 of the packed
// row spectra holds (X[0], X[W/2]), both real, with real factors E(0), E(W/2): it is combined
// component-wise.
#include "sfft_common.cuh"

struct ETabParams {
  const double* coeffs;
  cplx* E;  // [TK][2w+1][NC]
  int w, L, NC, W;
  const cplx* twW;
};

__global__ void __launch_bounds__(128) k_etable(ETabParams P) {
  const int kx = blockIdx.x * 128 + threadIdx.x;
  if (kx >= P.NC) return;
  const int S1 = 2 * P.w + 1;
  const int t = blockIdx.y / S1, vi = blockIdx.y % S1;
  const double* a = P.coeffs + (size_t)t * P.L + (size_t)vi * S1;
  cplx acc = cmake(0.0, 0.0);
  if (kx == 0) {
    for (int ui = 0; ui < S1; ++ui) {
      const int u = ui - P.w;
      acc.x += a[ui];
      acc.y += (u & 1) ? -a[ui] : a[ui];
    }
  } else {
    for (int ui = 0; ui < S1; ++ui) {
      const int u = ui - P.w;
      const cplx tw = ldg2(P.twW + ((kx * u) & (P.W - 1)));
      acc.x = fma(a[ui], tw.x, acc.x);
      acc.y = fma(a[ui], tw.y, acc.y);
    }
  }
  P.E[((size_t)t * S1 + vi) * P.NC + kx] = acc;
}

struct MixParams {
  const cplx* G;   // [DK+1][H][NC] row spectra of xi^p R
  const cplx* E;   // [TK][2w+1][NC]
  cplx* Mhat;      // [H][NC]
  int H, NC, DK, TK, KT;
  int monoK[SFFT_MAX_T][2];
};

#ifndef MIX_RY
#define MIX_RY 8   // output rows per thread
#endif
#ifndef MIX_MINB
#define MIX_MINB 2   // 2 CTAs per SM: up to 255 registers, no spills (3 CTAs at 168 registers spilled 250 bytes and were 2 % slower)
#endif
#define MIX_TH 128 // threads per block

// Register-tiled y-mixing (the eta^q factors of one xi power are folded by Horner's rule).  A thread owns one kx and MIX_RY consecutive output rows; per xi power p
// it loads the MIX_RY + 2w source rows of G_p once into registers, scales them by eta^q in place
// for q = 0..DK-p, and for every (q, v) applies one E value to all MIX_RY accumulators: one global
// (L1-resident) load per MIX_RY complex FMAs instead of two shared loads per FMA.  Lanes run
// along kx, so every load and store is a contiguous 512-byte segment.
// The packed column kx = 0 holds (X[0], X[W/2]), both real with real factors, and is combined
// component-wise by the extra x-block (four threads per row, fixed-order shuffle reduction).
template <int WK>
__global__ void __launch_bounds__(MIX_TH, MIX_MINB) k_mix(MixParams P) {
  constexpr int RY = MIX_RY, S1 = 2 * WK + 1, WIN = RY + 2 * WK;
  const int H = P.H, NC = P.NC, KT = P.KT;
  const int tid = threadIdx.x;
  const int rowsPerBlock = (MIX_TH / KT) * RY;
  const double invH = 1.0 / (double)H;
  if (blockIdx.x == gridDim.x - 1) {
    // ---- packed column (rowsPerBlock is a multiple of MIX_TH / 4, so the trip count is uniform)
    for (int r = tid >> 2; r < rowsPerBlock; r += MIX_TH / 4) {
      const int y = blockIdx.y * rowsPerBlock + r, part = tid & 3;
      const bool live = y < H;
      double ax = 0.0, ay = 0.0;
      if (live) {
        for (int idx = part; idx < P.TK * S1; idx += 4) {
          const int t = idx / S1, vi = idx - t * S1;
          int d = 0;                       // monomial t = (p, q) of the order "for d: for q <= d: p = d - q"
          while ((d + 1) * (d + 2) / 2 <= t) ++d;
          const int q = t - d * (d + 1) / 2, p = d - q;
          const int yy = (y - vi + WK + H) & (H - 1);
          const double eq = ipow((double)(2 * yy + 1 - H) * invH, q);
          const cplx e = P.E[(size_t)idx * NC];
          const cplx g = P.G[((size_t)p * H + yy) * NC];
          ax = fma(e.x * eq, g.x, ax);
          ay = fma(e.y * eq, g.y, ay);
        }
      }
      ax += __shfl_xor_sync(0xffffffffu, ax, 1);
      ay += __shfl_xor_sync(0xffffffffu, ay, 1);
      ax += __shfl_xor_sync(0xffffffffu, ax, 2);
      ay += __shfl_xor_sync(0xffffffffu, ay, 2);
      if (live && part == 0) P.Mhat[(size_t)y * NC] = cmake(ax, ay);
    }
    return;
  }
  const int kl = tid % KT, rg = tid / KT;
  const int kx = blockIdx.x * KT + kl;
  const int y0 = blockIdx.y * rowsPerBlock + rg * RY;
  if (y0 >= H) return;
  cplx acc[RY];
#pragma unroll
  for (int i = 0; i < RY; ++i) acc[i] = cmake(0.0, 0.0);
  double eta[WIN];   // eta of the window's source rows (each row's own coordinate, also when wrapped)
#pragma unroll
  for (int i = 0; i < WIN; ++i) {
    const int yy = (y0 - WK + i + H) & (H - 1);
    eta[i] = (double)(2 * yy + 1 - H) * invH;
  }
  // per xi power p: M += sum_v W_p(v, y - v) G_p[y - v],  W_p(v, y') = sum_q E_(p,q)[v] eta(y')^q
  // evaluated by Horner in eta, so a (v, row) pair costs one complex fma plus 2 (DK - p) real fmas
  for (int p = 0; p <= P.DK; ++p) {
    cplx g[WIN];
    const cplx* Gp = P.G + (size_t)p * H * NC + kx;
#pragma unroll
    for (int i = 0; i < WIN; ++i) {
      const int yy = (y0 - WK + i + H) & (H - 1);
      g[i] = Gp[(size_t)yy * NC];
    }
    const int nq = P.DK - p + 1;
    // E_(p,q) = monomial index d(d+1)/2 + q with d = p + q
    const cplx* E0 = P.E + (size_t)(p * (p + 1) / 2) * S1 * NC + kx;
    const cplx* E1 = P.E + (size_t)((p + 1) * (p + 2) / 2 + 1) * S1 * NC + kx;
    const cplx* E2 = P.E + (size_t)((p + 2) * (p + 3) / 2 + 2) * S1 * NC + kx;
    const cplx* E3 = P.E + (size_t)((p + 3) * (p + 4) / 2 + 3) * S1 * NC + kx;
    if (nq == 1) {
#pragma unroll
      for (int vi = 0; vi < S1; ++vi) {
        const cplx e0 = E0[(size_t)vi * NC];
#pragma unroll
        for (int i = 0; i < RY; ++i) cfma(acc[i], e0, g[i + 2 * WK - vi]);
      }
    } else if (nq == 2) {
#pragma unroll
      for (int vi = 0; vi < S1; ++vi) {
        const cplx e0 = E0[(size_t)vi * NC], e1 = E1[(size_t)vi * NC];
#pragma unroll
        for (int i = 0; i < RY; ++i) {
          const double h = eta[i + 2 * WK - vi];
          cfma(acc[i], cmake(fma(h, e1.x, e0.x), fma(h, e1.y, e0.y)), g[i + 2 * WK - vi]);
        }
      }
    } else if (nq == 3) {
#pragma unroll
      for (int vi = 0; vi < S1; ++vi) {
        const cplx e0 = E0[(size_t)vi * NC], e1 = E1[(size_t)vi * NC], e2 = E2[(size_t)vi * NC];
#pragma unroll
        for (int i = 0; i < RY; ++i) {
          const double h = eta[i + 2 * WK - vi];
          const cplx w = cmake(fma(h, fma(h, e2.x, e1.x), e0.x), fma(h, fma(h, e2.y, e1.y), e0.y));
          cfma(acc[i], w, g[i + 2 * WK - vi]);
        }
      }
    } else {
#pragma unroll
      for (int vi = 0; vi < S1; ++vi) {
        const cplx e0 = E0[(size_t)vi * NC], e1 = E1[(size_t)vi * NC], e2 = E2[(size_t)vi * NC], e3 = E3[(size_t)vi * NC];
#pragma unroll
        for (int i = 0; i < RY; ++i) {
          const double h = eta[i + 2 * WK - vi];
          const cplx w = cmake(fma(h, fma(h, fma(h, e3.x, e2.x), e1.x), e0.x), fma(h, fma(h, fma(h, e3.y, e2.y), e1.y), e0.y));
          cfma(acc[i], w, g[i + 2 * WK - vi]);
        }
      }
    }
  }
  if (kx != 0) {
#pragma unroll
    for (int i = 0; i < RY; ++i) P.Mhat[(size_t)(y0 + i) * NC + kx] = acc[i];
  }
}

// y-mixing for kernel half-widths above 5 (no register window: 2w+1 > 11 source rows per output row do not
// fit beside the accumulators).  Thread = one (y, kx); every (monomial, v) term is read from global memory
// (L1/L2-resident: neighbouring rows share their source rows).  Same sums as k_mix, monomial-major order.
__global__ void __launch_bounds__(MIX_TH) k_mix_gen(MixParams P, int w) {
  const int H = P.H, NC = P.NC, KT = P.KT, S1 = 2 * w + 1;
  const int kx = blockIdx.x * KT + threadIdx.x % KT;
  const int y = blockIdx.y * (MIX_TH / KT) + threadIdx.x / KT;
  if (y >= H || kx >= NC) return;
  const double invH = 1.0 / (double)H;
  cplx acc = cmake(0.0, 0.0);
  for (int t = 0; t < P.TK; ++t) {
    int d = 0;                       // monomial t = (p, q) of the order "for d: for q <= d: p = d - q"
    while ((d + 1) * (d + 2) / 2 <= t) ++d;
    const int q = t - d * (d + 1) / 2, p = d - q;
    for (int vi = 0; vi < S1; ++vi) {
      const int yy = (y - vi + w + H) & (H - 1);
      const double eq = ipow((double)(2 * yy + 1 - H) * invH, q);
      const cplx e = P.E[((size_t)t * S1 + vi) * NC + kx];
      const cplx g = P.G[((size_t)p * H + yy) * NC + kx];
      if (kx == 0) {                 // packed column (X[0], X[W/2]): both real with real factors, component-wise
        acc.x = fma(e.x * eq, g.x, acc.x);
        acc.y = fma(e.y * eq, g.y, acc.y);
      } else {
        cfma(acc, cmake(e.x * eq, e.y * eq), g);
      }
    }
  }
  P.Mhat[(size_t)y * NC + kx] = acc;
}

static sfft_status launch_mix_gen(const MixParams& MP, int w, cudaStream_t st) {
  dim3 grid((MP.NC + MP.KT - 1) / MP.KT, (MP.H + MIX_TH / MP.KT - 1) / (MIX_TH / MP.KT));
  k_mix_gen<<<grid, MIX_TH, 0, st>>>(MP, w);
  SFFT_LAUNCH_CHECK();
  return SFFT_OK;
}

template <int WK>
static sfft_status launch_mix_t(const MixParams& MP, cudaStream_t st) {
  const int rowsPerBlock = (MIX_TH / MP.KT) * MIX_RY;
  dim3 gm(MP.NC / MP.KT + 1, (MP.H + rowsPerBlock - 1) / rowsPerBlock);
  k_mix<WK><<<gm, MIX_TH, 0, st>>>(MP);
  SFFT_LAUNCH_CHECK();
  return SFFT_OK;
}

sfft_status sfft_launch_row_inv_sub(sfft_plan* p, const double* S, const double* c, double* D,
                                    cudaStream_t st, int* nl);

// row spectra of xi^p R (unmasked), p = 0..DK, into the row-pass scratch
sfft_status sfft_launch_subtract_rows(sfft_plan* p, const double* R, cudaStream_t st, int* nl) {
  ProfScope ps(p, 6, st);
  return sfft_launch_row_fwd(p, R, R, nullptr, false, p->T, p->NC, true, false, st, nl);
}

sfft_status sfft_launch_subtract(sfft_plan* p, const double* R, const double* S, const double* c,
                                 double* D, cudaStream_t st, int* nl) {
  // 1. row spectra of xi^p R: already there if sfft_subtract_prepare ran for this R
  sfft_status s;
  // (a pending prepare always has to finish first: it writes the same scratch)
  if (p->prepValid) SFFT_CUDA_TRY(cudaStreamWaitEvent(st, p->evPrep, 0));
  if (!(p->prepValid && p->prepR == R)) {
    s = sfft_launch_subtract_rows(p, R, st, nl);
    if (s != SFFT_OK) return s;
  }
  p->prepValid = 0;
  {
    ProfScope pmix(p, 7, st);
    // 2. x-phase table of the kernel coefficients
    ETabParams EP;
    EP.coeffs = c; EP.E = p->Etab; EP.w = p->w; EP.L = p->L; EP.NC = p->NC; EP.W = p->W; EP.twW = p->twW;
    dim3 ge((p->NC + 127) / 128, p->TK * (2 * p->w + 1));
    k_etable<<<ge, 128, 0, st>>>(EP);
    SFFT_LAUNCH_CHECK();
    ++*nl;
    // 3. y-mixing
    MixParams MP;
    MP.G = p->T; MP.E = p->Etab; MP.Mhat = p->Mhat; MP.H = p->H; MP.NC = p->NC;
    MP.DK = p->DK; MP.TK = p->TK;
    MP.KT = p->NC < 32 ? p->NC : 32;
    for (int t = 0; t < p->TK; ++t) { MP.monoK[t][0] = p->monoK[t][0]; MP.monoK[t][1] = p->monoK[t][1]; }
    switch (p->w) {
      case 0: s = launch_mix_t<0>(MP, st); break;
      case 1: s = launch_mix_t<1>(MP, st); break;
      case 2: s = launch_mix_t<2>(MP, st); break;
      case 3: s = launch_mix_t<3>(MP, st); break;
      case 4: s = launch_mix_t<4>(MP, st); break;
      case 5: s = launch_mix_t<5>(MP, st); break;
      default: s = launch_mix_gen(MP, p->w, st); break;   // w > 5
    }
  }
  if (s != SFFT_OK) return s;
  ++*nl;
  // 4. inverse rows + subtraction
  { ProfScope ps(p, 8, st); s = sfft_launch_row_inv_sub(p, S, c, D, st, nl); }
  return s;
}
