// Fused column pass + cross spectra + lag-pruned inverse along ky (north_star subsystems (2),(3);
// SURVEY.md §8(a) a2/a3) for H = 512*DR, DR in {2,4,8}: the spectra F never travel through HBM.
//
// One CTA owns two adjacent columns kx0, kx0+1 of the row spectra T and ONE residue class
// c = ky mod DR of the column frequencies.  With y = y' + 512 m, ky = DR k' + c:
//
//   F[DR k' + c] = sum_{y'<512} e^{-2 pi i y' k'/512} { e^{-2 pi i c y'/H} sum_{m<DR} w_DR^{c m} eta(y'+512m)^q T[y'+512m] }
//
// so every spectrum restricted to the class is ONE 512-point FFT of a decimated, twiddled column
// (phase A: load + decimate, phase B: FFT).  All nSpec spectra of both columns stay in shared
// memory (2*nSpec*8 KB = 112 KB at DK = 2: two CTAs per SM, one loading while the other computes).
// Phase C forms, for every pair (f,g), the class's share of
//   Y[dy][kx] = sum_ky conj(F_f) F_g e^{+2 pi i ky dy/H}
//             = sum_c e^{2 pi i c dy/H} sum_{b<64} e^{2 pi i b dy/512} Z_b[dy mod 8],
//   Z_b = 8-point inverse DFT over a of the products at k' = b + 64 a,
// with lanes = pairs (every shared-memory operand is a broadcast of <= nSpec distinct words) and
// warps = (column, quarter of the b range); phase D reduces the four quarters in a fixed order
// and writes the class's partial lag rows.  k_lag_idft adds the DR partials in class order.
//
// The 512-point transforms are warp-synchronous: one warp per sequence, 16 elements per lane, three
// in-place radix-8 Stockham passes (two butterflies per lane and pass) separated by __syncwarp
// only.  Shared-memory indices are XOR-swizzled, swz(n) = n ^ ((n >> 3) & 7), which makes every
// pass conflict free without padding; sequences are pitched 513 elements apart so that the same
// element of different spectra falls into different banks.
#include <math.h>
#include "fft_smem.cuh"

#define CX_N 512            // sequence length (k' range)
#define CX_PITCH 513        // sequence pitch in shared memory (complex elements)
#define CX_TH 256
#define CX_NW (CX_TH / 32)
#define CX_NBQ 4            // b-range quarters (warps per column in phase C)
#define CX_MAXSPEC (SFFT_MAX_T + 1)

struct ColxParams {
  const cplx* T;        // [nimg][NC/2+1][H][2] pair-major unpacked row spectra (columns 0..NC)
  cplx* Y;              // [DR][nPair][nLag][pitch] partial lag rows per residue class
  const PairDesc* pairs;
  int H, NC, pitchT, pitch, nLag, nPair, nSpec, nimg;
  int img_nq[SFFT_MAX_DEG + 2];                       // spectra fed by row image im: eta powers 0..nq-1
  int img_spec[SFFT_MAX_DEG + 2][SFFT_MAX_DEG + 1];   // their spectrum indices
  const cplx* twH;      // e^{-2 pi i m/H}
  const cplx* twP;      // per-pass tables of the 512-point FFT (fft_smem.cuh layout)
  int Dmax;             // lag half-range of the instantiation
};

// e^{-2 pi i bb i/512}, bb < 16, i = 1..10: the lag twiddles inside one quarter of the b range
// (fixed by the 512-point split, so one table serves every plan; written by sfft_colx_init).
// Held in constant memory: with the b loop unrolled they are immediate operands of the DFMAs.
#define CX_TWD 10
#ifndef CX_UNROLL
#define CX_UNROLL 4
#endif
constexpr int CXU = CX_UNROLL;   // unroll factor of the b loop in phase C
__constant__ cplx cx_twlag[16][CX_TWD];

__device__ __forceinline__ int cx_swz(int n) { return n ^ ((n >> 3) & 7); }
__host__ __device__ __forceinline__ int cx_col_stride(int nSpec) {
  const int n = nSpec * CX_PITCH;
  return n + ((4 - (n & 7)) & 7);
}

// sum_m w_DR^{c m} x[m]: the residue-c output of a DR-point forward DFT (c is CTA-uniform)
template <int DR>
__device__ __forceinline__ cplx cx_decim(const cplx* x, int c);
template <>
__device__ __forceinline__ cplx cx_decim<2>(const cplx* x, int c) {
  return c ? csub(x[0], x[1]) : cadd(x[0], x[1]);
}
__device__ __forceinline__ cplx cx_decim4(cplx x0, cplx x1, cplx x2, cplx x3, int c) {
  const bool odd = c & 1;
  const cplx e = odd ? csub(x0, x2) : cadd(x0, x2);
  const cplx o = odd ? csub(x1, x3) : cadd(x1, x3);
  switch (c & 3) {
    case 0: return cadd(e, o);
    case 1: return cadd(e, cmul_mi(o));   // w4 = -i
    case 2: return csub(e, o);
    default: return cadd(e, cmul_pi(o));
  }
}
template <>
__device__ __forceinline__ cplx cx_decim<4>(const cplx* x, int c) { return cx_decim4(x[0], x[1], x[2], x[3], c); }
template <>
__device__ __forceinline__ cplx cx_decim<8>(const cplx* x, int c) {
  const cplx e = cx_decim4(x[0], x[2], x[4], x[6], c);
  cplx o = cx_decim4(x[1], x[3], x[5], x[7], c);
  // w8^c, c < 8
  switch (c) {
    case 0: break;
    case 1: o = mul_w8_1<-1>(o); break;
    case 2: o = cmul_mi(o); break;
    case 3: o = mul_w8_3<-1>(o); break;
    case 4: o = cmake(-o.x, -o.y); break;
    case 5: o = cmake(-SFFT_SQRT1_2 * (o.x + o.y), SFFT_SQRT1_2 * (o.x - o.y)); break;   // e^{-5 pi i/4}
    case 6: o = cmul_pi(o); break;
    default: o = cmake(SFFT_SQRT1_2 * (o.x - o.y), SFFT_SQRT1_2 * (o.x + o.y)); break;   // e^{-7 pi i/4}
  }
  return cadd(e, o);
}

// One 512-point forward FFT, in place in shared memory, by one warp.
__device__ __forceinline__ void cx_warp_fft512(cplx* seq, int lane, const cplx* __restrict__ twP) {
  constexpr int NB = CX_N / 8;   // 64 butterflies per pass, two per lane
  cplx v[2][8];
  // pass 0 (NS = 1)
#pragma unroll
  for (int m = 0; m < 2; ++m) {
    const int j = lane + 32 * m, pj = cx_swz(j);
#pragma unroll
    for (int r = 0; r < 8; ++r) v[m][r] = seq[pj + r * NB];
  }
  __syncwarp();
#pragma unroll
  for (int m = 0; m < 2; ++m) {
    const int j = lane + 32 * m;
    Dft<8, -1>::run(v[m]);
#pragma unroll
    for (int r = 0; r < 8; ++r) seq[8 * j + (r ^ (j & 7))] = v[m][r];
  }
  __syncwarp();
  // pass 1 (NS = 8)
  {
    const cplx* tw = twP + fft_tw_off(CX_N, 1);
#pragma unroll
    for (int m = 0; m < 2; ++m) {
      const int j = lane + 32 * m, pj = cx_swz(j);
#pragma unroll
      for (int r = 0; r < 8; ++r) v[m][r] = seq[pj + r * NB];
    }
    __syncwarp();
#pragma unroll
    for (int m = 0; m < 2; ++m) {
      const int j = lane + 32 * m, k = j & 7;
      cplx t[8];
#pragma unroll
      for (int r = 1; r < 8; ++r) t[r] = ldg2(tw + (r - 1) * 8 + k);
#pragma unroll
      for (int r = 1; r < 8; ++r) v[m][r] = cmul(v[m][r], t[r]);
      Dft<8, -1>::run(v[m]);
      const int o = (j - k) * 8;   // multiple of 64: bits 3..5 of o + 8r + k are r
#pragma unroll
      for (int r = 0; r < 8; ++r) seq[o + 8 * r + (k ^ r)] = v[m][r];
    }
    __syncwarp();
  }
  // pass 2 (NS = 64)
  {
    const cplx* tw = twP + fft_tw_off(CX_N, 2);
#pragma unroll
    for (int m = 0; m < 2; ++m) {
      const int j = lane + 32 * m, pj = cx_swz(j);
#pragma unroll
      for (int r = 0; r < 8; ++r) v[m][r] = seq[pj + r * NB];
    }
    __syncwarp();
#pragma unroll
    for (int m = 0; m < 2; ++m) {
      const int j = lane + 32 * m, pj = cx_swz(j);
      cplx t[8];
#pragma unroll
      for (int r = 1; r < 8; ++r) t[r] = ldg2(tw + (r - 1) * 64 + j);
#pragma unroll
      for (int r = 1; r < 8; ++r) v[m][r] = cmul(v[m][r], t[r]);
      Dft<8, -1>::run(v[m]);
#pragma unroll
      for (int r = 0; r < 8; ++r) seq[pj + 64 * r] = v[m][r];   // X[j + 64 r], natural order
    }
  }
}

// D = lag half-range of the instantiation (>= the largest half-range of any pair).
template <int DR, int D>
__global__ void __launch_bounds__(CX_TH, 2) k_colx(ColxParams P) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx* sq = reinterpret_cast<cplx*>(smem_raw);   // [2*nSpec][CX_PITCH]; sequence = col*nSpec + spec
  const int tid = threadIdx.x, lane = tid & 31, wrp = tid >> 5;
  const int c = blockIdx.x % DR;                   // residue class of ky
  const int kx0 = (blockIdx.x / DR) * 2;
  const int H = P.H, nSpec = P.nSpec;
  const double invH = 1.0 / (double)H;
  // column 1's sequences start 4 (mod 8) elements after column 0's: the two columns of phase A's
  // quarter-warp stores fall into disjoint bank groups
  const int colStride = cx_col_stride(nSpec);

  // ---- phase A: load the two columns of every row image, decimate to the class, twiddle -------
  constexpr int KB = 16 / DR > 4 ? 4 : 16 / DR;    // items per thread and batch (KB*DR loads in flight)
  const double deta = (double)(2 * CX_N) * invH;   // eta(y' + 512 m) = eta(y') + m * deta
  for (int im = 0; im < P.nimg; ++im) {
    const cplx* Tim = P.T + ((size_t)im * (P.NC / 2 + 1) + (kx0 >> 1)) * H * 2;
    const int nq = P.img_nq[im];
#pragma unroll 1
    for (int k0 = 0; k0 < CX_N * 2 / CX_TH; k0 += KB) {
      cplx x[KB][DR];
#pragma unroll
      for (int k = 0; k < KB; ++k) {
        const cplx* src = Tim + tid + CX_TH * (k0 + k);   // element (yp, col) at 2*yp + col
#pragma unroll
        for (int m = 0; m < DR; ++m) x[k][m] = src[CX_N * 2 * m];
      }
#pragma unroll
      for (int k = 0; k < KB; ++k) {
        const int i = tid + CX_TH * (k0 + k), col = i & 1, yp = i >> 1;
        const cplx tw = ldg2(P.twH + c * yp);       // e^{-2 pi i c y'/H}; c*yp < H
        const double eta0 = (double)(2 * yp + 1 - H) * invH;
        cplx* dst = sq + (size_t)col * colStride + cx_swz(yp);
        for (int q = 0; q < nq; ++q) {
          if (q > 0) {
#pragma unroll
            for (int m = 0; m < DR; ++m) x[k][m] = cscale(x[k][m], eta0 + (double)m * deta);
          }
          cplx s = cx_decim<DR>(x[k], c);
          if (c) s = cmul(s, tw);
          dst[(size_t)P.img_spec[im][q] * CX_PITCH] = s;
        }
      }
    }
  }
  __syncthreads();

  // ---- phase B: one warp per sequence ---------------------------------------------------------
  for (int sidx = wrp; sidx < 2 * nSpec; sidx += CX_NW)
    cx_warp_fft512(sq + (size_t)(sidx / nSpec) * colStride + (size_t)(sidx % nSpec) * CX_PITCH, lane, P.twP);
  __syncthreads();

  // ---- phase C: cross products + pruned inverse; lanes = pairs, warps = (column, b quarter) ----
  const int col = wrp / CX_NBQ, bq = wrp % CX_NBQ;
  constexpr int NBW = (CX_N / 8) / CX_NBQ;   // 16 b values per warp
  cplx* red = sq;                              // phase D scratch aliases the spectra (after a barrier)
  {
    const int pg = 0;          // the fused path is used only when all pairs fit the 32 lanes
    const int pair = pg + lane;
    const bool has_pair = pair < P.nPair;
    const PairDesc pd = P.pairs[has_pair ? pair : 0];
    const cplx* pa = sq + (size_t)col * colStride + (size_t)pd.fa * CX_PITCH;
    const cplx* pb = sq + (size_t)col * colStride + (size_t)pd.fb * CX_PITCH;
    cplx acc[2 * D + 1];
#pragma unroll
    for (int i = 0; i < 2 * D + 1; ++i) acc[i] = cmake(0.0, 0.0);
#pragma unroll CXU
    for (int bb = 0; bb < NBW; ++bb) {
      const int pbv = cx_swz(bq * NBW + bb);
      cplx x[8];
#pragma unroll
      for (int a = 0; a < 8; ++a) x[a] = cmulc(pa[pbv + 64 * a], pb[pbv + 64 * a]);
      Dft<8, +1>::run(x);
      acc[D] = cadd(acc[D], x[0]);
#pragma unroll
      for (int i = 1; i <= D; ++i) {
        const cplx t = cx_twlag[bb][i - 1];                // e^{-2 pi i bb i/512}
        cfmac(acc[D + i], t, x[i & 7]);                    // += e^{+...} * Z[i mod 8]
        cfma(acc[D - i], t, x[(8 - (i & 7)) & 7]);         // += e^{-...} * Z[-i mod 8]
      }
    }
    // quarter phase e^{2 pi i (16 bq) dy/512} and class phase e^{2 pi i c dy/H}
#pragma unroll
    for (int i = 1; i <= D; ++i) {
      const cplx t = cmul(ldg2(P.twH + ((bq * i * (H / 32)) & (H - 1))), ldg2(P.twH + c * i));
      acc[D + i] = cmulc(t, acc[D + i]);
      acc[D - i] = cmul(t, acc[D - i]);
    }
    // ---- phase D: fixed-order reduction over the b quarters, then the partial lag rows --------
    __syncthreads();   // every warp has finished reading the spectra (or the previous group's red)
#pragma unroll
    for (int i = 0; i < 2 * D + 1; ++i) red[((size_t)(col * CX_NBQ + bq) * (2 * D + 1) + i) * 32 + lane] = acc[i];
    __syncthreads();
    for (int o = tid; o < 2 * 32 * (2 * D + 1); o += CX_TH) {
      const int oc = o & 1, op = (o >> 1) & 31, oi = o >> 6;
      const int opair = pg + op;
      if (opair >= P.nPair || kx0 + oc > P.NC) continue;
      const int Dp = P.pairs[opair].D, dy = oi - D;
      if (dy < -Dp || dy > Dp) continue;
      cplx sum = cmake(0.0, 0.0);
#pragma unroll
      for (int q = 0; q < CX_NBQ; ++q) sum = cadd(sum, red[((size_t)(oc * CX_NBQ + q) * (2 * D + 1) + oi) * 32 + op]);
      P.Y[(((size_t)c * P.nPair + opair) * P.nLag + (dy + Dp)) * P.pitch + kx0 + oc] = sum;
    }
  }
}

template <int DR, int D>
static sfft_status launch_colx_t(const ColxParams& P, cudaStream_t st) {
  size_t smem = (size_t)2 * cx_col_stride(P.nSpec) * sizeof(cplx);
  const size_t red = (size_t)2 * CX_NBQ * (2 * D + 1) * 32 * sizeof(cplx);
  if (smem < red) smem = red;
  SFFT_CUDA_TRY(cudaFuncSetAttribute(k_colx<DR, D>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  k_colx<DR, D><<<(P.NC / 2 + 1) * DR, CX_TH, smem, st>>>(P);
  SFFT_LAUNCH_CHECK();
  return SFFT_OK;
}

template <int DR>
static sfft_status launch_colx_d(const ColxParams& P, cudaStream_t st) {
  switch (P.Dmax) {
    case 1: return launch_colx_t<DR, 1>(P, st);
    case 2: return launch_colx_t<DR, 2>(P, st);
    case 4: return launch_colx_t<DR, 4>(P, st);
    case 6: return launch_colx_t<DR, 6>(P, st);
    case 8: return launch_colx_t<DR, 8>(P, st);
    case 10: return launch_colx_t<DR, 10>(P, st);
    default: return SFFT_ERR_UNSUPPORTED;
  }
}

// lag half-range the kernel is instantiated with for kernel half-width w
int sfft_colx_dinst(int w) { return w == 0 ? 1 : 2 * w; }

bool sfft_colx_supported(int H, int nPair) { return (H == 1024 || H == 2048 || H == 4096) && nPair <= 32; }

// one-time upload of the constant lag-twiddle table (same values for every plan)
sfft_status sfft_colx_init() {
  cplx h[16][CX_TWD];
  const long double twopi = 6.283185307179586476925286766559005768L;
  for (int bb = 0; bb < 16; ++bb)
    for (int i = 1; i <= CX_TWD; ++i) {
      const int num = (bb * i) % 512;
      const long double ang = -twopi * (long double)num / 512.0L;
      h[bb][i - 1] = num == 0 ? cmake(1.0, 0.0) : (num == 128 ? cmake(0.0, -1.0) : cmake((double)cosl(ang), (double)sinl(ang)));
    }
  SFFT_CUDA_TRY(cudaMemcpyToSymbol(cx_twlag, h, sizeof(h)));
  return SFFT_OK;
}

sfft_status sfft_launch_colx(sfft_plan* p, cudaStream_t st, int* nl) {
  ColxParams P;
  P.T = p->T; P.Y = p->Y; P.pairs = p->d_pairs; P.H = p->H; P.NC = p->NC; P.pitchT = 0;
  P.pitch = p->pitch; P.nLag = p->nLag; P.nPair = p->nPair; P.nSpec = p->nSpec; P.nimg = p->nRowImg;
  for (int im = 0; im <= p->DK; ++im) P.img_nq[im] = 0;
  for (int t = 0; t < p->TK; ++t) {   // spectrum t = (p,q) comes from row image p with eta^q
    const int im = p->monoK[t][0], q = p->monoK[t][1];
    P.img_spec[im][q] = t;
    if (q + 1 > P.img_nq[im]) P.img_nq[im] = q + 1;
  }
  P.img_nq[p->DK + 1] = 1; P.img_spec[p->DK + 1][0] = p->TK;   // S~
  P.twH = p->twH; P.twP = p->twP512; P.Dmax = sfft_colx_dinst(p->w);
  ++*nl;
  switch (p->H / CX_N) {
    case 2: return launch_colx_d<2>(P, st);
    case 4: return launch_colx_d<4>(P, st);
    case 8: return launch_colx_d<8>(P, st);
    default: return SFFT_ERR_UNSUPPORTED;
  }
}
