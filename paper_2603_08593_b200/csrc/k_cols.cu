// Forward column pass of the batched 2-D real FFT (north_star subsystem (2)).
//
// Input : T[src][y][kx]  row spectra of the xi-weighted images (kx in [0,NC), column 0 packed
//         as X[0] + i X[W/2]).
// Output: F[spec][ky][kx] = sum_y eta(y)^q T[src][y][kx] e^{-2 pi i ky y/H}, kx in [0,NC], the
//         eta^q factor of monomial (p,q) being applied here (it commutes with the row pass).
//         The packed column is separated after its transform: with Z = F0 + i FN and F0, FN
//         Hermitian in ky,  F0[ky] = (Z[ky] + conj Z[-ky])/2,  FN[ky] = (Z[ky] - conj Z[-ky])/(2i);
//         FN is stored as column NC of the pitch-padded spectrum.
//
// One CTA transforms NCOL adjacent columns of one source image and loops over the eta powers that
// source feeds (up to DK+1 spectra per load pattern).  The first radix pass takes its inputs
// straight from global memory (each thread's 16 loads are independent and in flight together;
// adjacent lanes are adjacent columns, so a warp touches whole 32/64-byte segments) and the last
// pass writes its outputs straight to global memory, so shared memory only carries the
// exchanges between passes.  Small CTAs (2 columns at H = 2048) leave room for two or three per
// SM, which overlaps one CTA's loads and stores with another's butterflies.
#include "fft_smem.cuh"

#define COL_MAXGRP (2 * (SFFT_MAX_DEG + 1) + 1)

struct ColFwdParams {
  const cplx* T;
  cplx* F;
  int H, NC, pitch, ncol, skew;
  int ngrp;
  int grp_src[COL_MAXGRP];                    // source row-pass image
  int grp_n[COL_MAXGRP];                      // spectra produced from it
  int grp_spec[COL_MAXGRP][SFFT_MAX_DEG + 1];  // their spectrum indices
  int grp_q[COL_MAXGRP][SFFT_MAX_DEG + 1];     // and eta powers
  const cplx* twP;                            // per-pass twiddle tables for length H
};

template <int HH, int MINB>
__global__ void __launch_bounds__(HH >= 4096 ? 512 : 256, MINB) k_col_fwd(ColFwdParams P) {
  using C = FftCfg<HH>;
  constexpr int EPT = C::EPT;
  constexpr int NB0 = HH / EPT;                          // first-pass butterflies per column
  constexpr int RL = fft_radix(HH, C::NPASS - 1);        // last radix
  constexpr int NBL = HH / RL, ITL = EPT / RL;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx* s = reinterpret_cast<cplx*>(smem_raw);
  const int tid = threadIdx.x, nth = blockDim.x;
  const int ncol = P.ncol;
  const int seq_stride = C::SEQ_STRIDE + P.skew;
  const int kx0 = blockIdx.x * ncol;
  const int g = blockIdx.y;
  const double invH = 1.0 / (double)HH;
  int c0, j0;
  fft_map<NB0, true, 1>(tid, 0, nth, ncol, c0, j0);
  const cplx* in = P.T + (size_t)P.grp_src[g] * HH * P.NC + kx0 + c0;
  const int nspec = P.grp_n[g];
  for (int is = 0; is < nspec; ++is) {
    const int q = P.grp_q[g][is];
    cplx v[EPT];
#pragma unroll
    for (int r = 0; r < EPT; ++r) v[r] = in[(size_t)(j0 + r * NB0) * P.NC];
    if (q > 0) {
#pragma unroll
      for (int r = 0; r < EPT; ++r) {
        const double e = ipow((double)(2 * (j0 + r * NB0) + 1 - HH) * invH, q);
        v[r].x *= e;
        v[r].y *= e;
      }
    }
    fft_regs_to_regs<HH, -1, true>(v, s, tid, nth, ncol, P.twP, seq_stride);
    cplx* out = P.F + (size_t)P.grp_spec[g][is] * HH * P.pitch + kx0;
    if (kx0 != 0) {
#pragma unroll
      for (int m = 0; m < ITL; ++m) {
        int c, j;
        fft_map<NBL, true, 1>(tid, m, nth, ncol, c, j);
#pragma unroll
        for (int r = 0; r < RL; ++r) out[(size_t)(j + r * NBL) * P.pitch + c] = v[m * RL + r];
      }
      if (C::NPASS > 1) __syncthreads();  // the next spectrum's first pass overwrites s
    } else {
      // CTA holding the packed column: columns c > 0 go out directly, column 0 is separated
      // into the DC and Nyquist columns through shared memory
      if (C::NPASS > 1) __syncthreads();  // every thread has finished reading s
#pragma unroll
      for (int m = 0; m < ITL; ++m) {
        int c, j;
        fft_map<NBL, true, 1>(tid, m, nth, ncol, c, j);
#pragma unroll
        for (int r = 0; r < RL; ++r) {
          const int ky = j + r * NBL;
          if (c == 0) s[C::phys(ky)] = v[m * RL + r];
          else out[(size_t)ky * P.pitch + c] = v[m * RL + r];
        }
      }
      __syncthreads();
      for (int ky = tid; ky < HH; ky += nth) {
        const cplx z = s[C::phys(ky)];
        const cplx zm = cconj(s[C::phys((HH - ky) & (HH - 1))]);
        out[(size_t)ky * P.pitch] = cscale(cadd(z, zm), 0.5);
        out[(size_t)ky * P.pitch + P.NC] = cmul_mi(cscale(csub(z, zm), 0.5));
      }
      __syncthreads();
    }
  }
}

template <int HH>
static sfft_status launch_col_fwd_t(ColFwdParams& P, cudaStream_t st) {
  using C = FftCfg<HH>;
  // threads per column = HH/EPT; aim for 256-thread CTAs, at least 2 columns (32-byte segments)
  int ncol = 256 * C::EPT / HH;
  if (ncol < 2) ncol = 2;
  if (ncol > P.NC) ncol = P.NC;
  P.ncol = ncol;
  P.skew = ncol >= 8 ? 1 : 8 / ncol;   // keeps the column-interleaved accesses conflict free
  const int nth = ncol * HH / C::EPT;
  // H = 4096 needs 256 threads per column: one 512-thread CTA per SM
  const size_t smem = (size_t)ncol * (C::SEQ_STRIDE + P.skew) * sizeof(cplx);
  constexpr int MINB = HH >= 4096 ? 1 : 2;
  SFFT_CUDA_TRY(cudaFuncSetAttribute(k_col_fwd<HH, MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  dim3 grid(P.NC / ncol, P.ngrp);
  k_col_fwd<HH, MINB><<<grid, nth, smem, st>>>(P);
  SFFT_LAUNCH_CHECK();
  return SFFT_OK;
}

sfft_status sfft_launch_col_fwd(sfft_plan* p, cudaStream_t st, int* nl) {
  ColFwdParams P;
  P.T = p->T; P.F = p->F; P.H = p->H; P.NC = p->NC; P.pitch = p->pitch; P.twP = p->twPH;
  // spectra order: R~ monomials (TK), S~; row-pass images: R~ xi^p (DK+1), S~.
  // Groups are listed heaviest first (most eta powers per source).
  int n = 0;
  auto add_group = [&](int src, int pxi, int deg, int spec0, const int (*mono)[2], int nmono) {
    int k = 0;
    for (int t = 0; t < nmono; ++t)
      if (mono[t][0] == pxi) { P.grp_spec[n][k] = spec0 + t; P.grp_q[n][k] = mono[t][1]; ++k; }
    (void)deg;
    P.grp_src[n] = src; P.grp_n[n] = k; ++n;
  };
  for (int pxi = 0; pxi <= p->DK; ++pxi) {
    add_group(pxi, pxi, p->DK, 0, p->monoK, p->TK);
    if (pxi == 0) { P.grp_src[n] = p->DK + 1; P.grp_n[n] = 1; P.grp_spec[n][0] = p->TK; P.grp_q[n][0] = 0; ++n; }
  }
  P.ngrp = n;
  ++*nl;
  switch (p->H) {
    case 16: return launch_col_fwd_t<16>(P, st);
    case 32: return launch_col_fwd_t<32>(P, st);
    case 64: return launch_col_fwd_t<64>(P, st);
    case 128: return launch_col_fwd_t<128>(P, st);
    case 256: return launch_col_fwd_t<256>(P, st);
    case 512: return launch_col_fwd_t<512>(P, st);
    case 1024: return launch_col_fwd_t<1024>(P, st);
    case 2048: return launch_col_fwd_t<2048>(P, st);
    case 4096: return launch_col_fwd_t<4096>(P, st);
    default: return SFFT_ERR_UNSUPPORTED;
  }
}
