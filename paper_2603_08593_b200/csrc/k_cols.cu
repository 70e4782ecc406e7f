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
// One CTA transforms NCOL adjacent columns of one spectrum in shared memory.
#include "fft_smem.cuh"

struct ColFwdParams {
  const cplx* T;
  cplx* F;
  int H, NC, pitch, ncol;
  int src[2 * SFFT_MAX_T + 1];
  int qeta[2 * SFFT_MAX_T + 1];
  const cplx* twH;
};

template <int HH>
__global__ void __launch_bounds__(512) k_col_fwd(ColFwdParams P) {
  using C = FftCfg<HH>;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx* s = reinterpret_cast<cplx*>(smem_raw);
  const int tid = threadIdx.x, nth = blockDim.x;
  const int ncol = P.ncol;
  const int skew = ncol >= 8 ? 1 : 8 / ncol;       // keeps the column-interleaved staging conflict free
  const int seq_stride = C::SEQ_STRIDE + skew;
  const int kx0 = blockIdx.x * ncol;
  const int spec = blockIdx.y;
  const int q = P.qeta[spec];
  const cplx* in = P.T + (size_t)P.src[spec] * HH * P.NC + kx0;
  const double invH = 1.0 / (double)HH;
  for (int idx = tid; idx < ncol * HH; idx += nth) {
    const int c = idx % ncol, y = idx / ncol;
    cplx v = in[(size_t)y * P.NC + c];
    if (q > 0) {
      const double e = ipow((double)(2 * y + 1 - HH) * invH, q);
      v.x *= e;
      v.y *= e;
    }
    s[c * seq_stride + C::phys(y)] = v;
  }
  __syncthreads();
  fft_smem<HH, -1>(s, tid, nth, P.twH, seq_stride);
  cplx* out = P.F + (size_t)spec * HH * P.pitch + kx0;
  for (int idx = tid; idx < ncol * HH; idx += nth) {
    const int c = idx % ncol, ky = idx / ncol;
    const cplx z = s[c * seq_stride + C::phys(ky)];
    if (kx0 + c == 0) {
      const cplx zm = cconj(s[C::phys((HH - ky) & (HH - 1))]);
      out[(size_t)ky * P.pitch] = cscale(cadd(z, zm), 0.5);
      out[(size_t)ky * P.pitch + P.NC] = cmul_mi(cscale(csub(z, zm), 0.5));
    } else {
      out[(size_t)ky * P.pitch + c] = z;
    }
  }
}

template <int HH>
static sfft_status launch_col_fwd_t(ColFwdParams& P, int nspec, cudaStream_t st) {
  using C = FftCfg<HH>;
  int ncol = 256 * C::EPT / HH;
  if (ncol < 4) ncol = 4;
  if (HH >= 4096) ncol = 2;
  if (ncol > P.NC) ncol = P.NC;
  P.ncol = ncol;
  const int nth = ncol * HH / C::EPT;
  const int skew = ncol >= 8 ? 1 : 8 / ncol;
  const size_t smem = (size_t)ncol * (C::SEQ_STRIDE + skew) * sizeof(cplx);
  SFFT_CUDA_TRY(cudaFuncSetAttribute(k_col_fwd<HH>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  dim3 grid(P.NC / ncol, nspec);
  k_col_fwd<HH><<<grid, nth, smem, st>>>(P);
  SFFT_LAUNCH_CHECK();
  return SFFT_OK;
}

sfft_status sfft_launch_col_fwd(sfft_plan* p, cudaStream_t st, int* nl) {
  ColFwdParams P;
  P.T = p->T; P.F = p->F; P.H = p->H; P.NC = p->NC; P.pitch = p->pitch; P.twH = p->twH;
  // spectra order: R~ monomials (TK), S~, Psi monomials (TB)
  int n = 0;
  for (int t = 0; t < p->TK; ++t) { P.src[n] = p->monoK[t][0]; P.qeta[n] = p->monoK[t][1]; ++n; }
  P.src[n] = p->DK + 1; P.qeta[n] = 0; ++n;
  for (int t = 0; t < p->TB; ++t) { P.src[n] = p->DK + 2 + p->monoB[t][0]; P.qeta[n] = p->monoB[t][1]; ++n; }
  ++*nl;
  switch (p->H) {
    case 16: return launch_col_fwd_t<16>(P, n, st);
    case 32: return launch_col_fwd_t<32>(P, n, st);
    case 64: return launch_col_fwd_t<64>(P, n, st);
    case 128: return launch_col_fwd_t<128>(P, n, st);
    case 256: return launch_col_fwd_t<256>(P, n, st);
    case 512: return launch_col_fwd_t<512>(P, n, st);
    case 1024: return launch_col_fwd_t<1024>(P, n, st);
    case 2048: return launch_col_fwd_t<2048>(P, n, st);
    case 4096: return launch_col_fwd_t<4096>(P, n, st);
    default: return SFFT_ERR_UNSUPPORTED;
  }
}
