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
  int H, NC, w, DK, TK, KT;
};

#define MIX_YT 32

__global__ void __launch_bounds__(256) k_mix(MixParams P) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int KT = P.KT, w = P.w, S1 = 2 * w + 1, H = P.H, NC = P.NC;
  const int nrow = MIX_YT + 2 * w;
  cplx* Gs = reinterpret_cast<cplx*>(smem_raw);           // [DK+1][nrow][KT]
  cplx* Es = Gs + (size_t)(P.DK + 1) * nrow * KT;         // [TK][S1][KT]
  const int kx0 = blockIdx.x * KT, y0 = blockIdx.y * MIX_YT;
  const int tid = threadIdx.x;
  for (int e = tid; e < (P.DK + 1) * nrow * KT; e += 256) {
    const int kl = e % KT, ri = (e / KT) % nrow, p = e / (KT * nrow);
    const int yy = (y0 - w + ri + H) & (H - 1);
    Gs[e] = P.G[((size_t)p * H + yy) * NC + kx0 + kl];
  }
  for (int e = tid; e < P.TK * S1 * KT; e += 256) {
    const int kl = e % KT, r = e / KT;
    Es[e] = P.E[(size_t)r * NC + kx0 + kl];
  }
  __syncthreads();
  const int kl = tid % KT, rg = tid / KT;
  const int nrg = 256 / KT;                 // row groups
  const int rows_per = MIX_YT / nrg;        // rows per thread
  const double invH = 1.0 / (double)H;
  const bool packed = (kx0 + kl) == 0;
  for (int rr = 0; rr < rows_per; ++rr) {
    const int yi = rg * rows_per + rr;
    cplx acc = cmake(0.0, 0.0);
    for (int vi = 0; vi < S1; ++vi) {
      const int ri = yi + 2 * w - vi;  // source row y - v, v = vi - w, as an index into the tile
      const int yy = (y0 - w + ri + H) & (H - 1);
      const double eta = (double)(2 * yy + 1 - H) * invH;
      for (int p = 0; p <= P.DK; ++p) {
        // c_p = sum_q E_(p,q)[v] eta^q (Horner, highest q first); t(p,q) = d(d+1)/2 + q, d = p+q
        cplx c = cmake(0.0, 0.0);
        for (int q = P.DK - p; q >= 0; --q) {
          const int d = p + q;
          const cplx e = Es[((d * (d + 1) / 2 + q) * S1 + vi) * KT + kl];
          c.x = fma(c.x, eta, e.x);
          c.y = fma(c.y, eta, e.y);
        }
        const cplx g = Gs[((size_t)p * nrow + ri) * KT + kl];
        if (packed) {
          acc.x = fma(c.x, g.x, acc.x);
          acc.y = fma(c.y, g.y, acc.y);
        } else {
          cfma(acc, c, g);
        }
      }
    }
    P.Mhat[(size_t)(y0 + yi) * NC + kx0 + kl] = acc;
  }
}

sfft_status sfft_launch_row_inv_sub(sfft_plan* p, const double* S, const double* c, double* D,
                                    cudaStream_t st, int* nl);

sfft_status sfft_launch_subtract(sfft_plan* p, const double* R, const double* S, const double* c,
                                 double* D, cudaStream_t st, int* nl) {
  // 1. row spectra of xi^p R (unmasked), p = 0..DK, into the row-pass scratch
  RowImage imgs[SFFT_MAX_DEG + 1];
  for (int q = 0; q <= p->DK; ++q) { imgs[q].src = 0; imgs[q].pxi = q; imgs[q].masked = 0; }
  sfft_status s;
  { ProfScope ps(p, 6, st); s = sfft_launch_row_fwd(p, R, S, nullptr, imgs, p->DK + 1, p->T, false, st, nl); }
  if (s != SFFT_OK) return s;
  ProfScope* pmix = new ProfScope(p, 7, st);
  // 2. x-phase table of the kernel coefficients
  ETabParams EP;
  EP.coeffs = c; EP.E = p->Etab; EP.w = p->w; EP.L = p->L; EP.NC = p->NC; EP.W = p->W; EP.twW = p->twW;
  dim3 ge((p->NC + 127) / 128, p->TK * (2 * p->w + 1));
  k_etable<<<ge, 128, 0, st>>>(EP);
  SFFT_LAUNCH_CHECK();
  ++*nl;
  // 3. y-mixing
  MixParams MP;
  MP.G = p->T; MP.E = p->Etab; MP.Mhat = p->Mhat; MP.H = p->H; MP.NC = p->NC; MP.w = p->w;
  MP.DK = p->DK; MP.TK = p->TK;
  int KT = 32;
  if (KT > p->NC) KT = p->NC;
  auto need = [&](int kt) {
    return ((size_t)(p->DK + 1) * (MIX_YT + 2 * p->w) + (size_t)p->TK * (2 * p->w + 1)) * kt * sizeof(cplx);
  };
  while (KT > 8 && need(KT) > 200 * 1024) KT >>= 1;
  MP.KT = KT;
  const size_t smem = need(KT);
  SFFT_CUDA_TRY(cudaFuncSetAttribute(k_mix, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  const int yt = p->H < MIX_YT ? p->H : MIX_YT;
  if (yt != MIX_YT) return SFFT_ERR_UNSUPPORTED;
  dim3 gm(p->NC / KT, p->H / MIX_YT);
  k_mix<<<gm, 256, smem, st>>>(MP);
  delete pmix;
  SFFT_LAUNCH_CHECK();
  ++*nl;
  // 4. inverse rows + subtraction
  { ProfScope ps(p, 8, st); s = sfft_launch_row_inv_sub(p, S, c, D, st, nl); }
  return s;
}
