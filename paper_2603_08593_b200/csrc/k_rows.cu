// Row-direction kernels.
//
//  k_row2_fwd  : (a1)+(a2 first pass) -- generation of the polynomial-weighted, masked images
//                m xi^p R, m S fused into the first (row, R2C) pass of the 2-D FFT, plus the fused
//                fp64 row reductions sum_x m xi^a, sum_x m xi^a S and sum_x m xi^a R
//                (north_star subsystems (1),(2)).  The eta^q factor of a
//                monomial is a function of y only, so it commutes with the row transform and is
//                applied by the column pass: only DK+1 (not T_K) row transforms of R are needed.
//  k_row_inv_sub: (a6 last pass) -- C2R row transform of the mixed row spectra, fused with
//                D = S - M - B (north_star subsystem (6)).
//
// Real rows of length W are transformed as W/2-point complex FFTs of z[j] = x[2j] + i x[2j+1]
// with the standard split/merge post-(pre-)processing.  Two output layouts: the row-group layout of
// the fused build path (see k_row2_fwd) and the row-major packed one, T[y][kx], kx < W/2, whose
// column 0 packs the two real bins, T[y][0] = X[0] + i X[W/2] (generic build path, sfft_subtract).
#include "fft_smem.cuh"

struct RowFwdParams {
  const double* R;
  const double* S;
  const unsigned char* mask;   // applied when non-NULL
  int H, W;
  int nR;        // images 0..nR-1 are xi^p R, p = image index
  int withS;     // image nR is S (weight 1)
  cplx* T;       // colT = 0: [nimg][H][pitchT];  colT = 1: [nimg][H/G][NC+1][G]
  int pitchT;    // row pitch of T in complex elements
  int packed;    // 1: T[y][0] = X[0] + i X[W/2];  0: T[y][0] = X[0], T[y][NC] = X[W/2]
  int colT;      // 1 (unpacked only): row-group layout T[img][y/G][kx][y%G], G = SFFT_T_G, kx in [0, NC]; written by k_row2_fwd, read by k_colb
  const cplx* twP;   // per-pass twiddle tables for length NC
  const cplx* twW;
  int moments, DB, nMomA, nMomS, nMomR;
  double fullA[2 * SFFT_MAX_DEG + 1];   // sum over a whole row of xi^a
  double* rowMom;  // [nMomA + nMomS + nMomR][H]
};

#define ROW_NMA (2 * SFFT_MAX_DEG + 1)   // most mask moments
// streaming (evict-first) accesses for the bulk data keep the twiddle tables resident in L1
#define SFFT_ROW_STREAM 1
#ifdef SFFT_ROW_STREAM
#define ROW_LD(p) __ldcs(p)
#define ROW_ST(p, v) __stcs(p, v)
#else
#define ROW_LD(p) (*(p))
#define ROW_ST(p, v) (*(p) = (v))
#endif
#ifndef SFFT_ROW_AHEAD
#define SFFT_ROW_AHEAD 48   // k_row2_fwd: CTA-loads of row pairs between a CTA and the pair it prefetches into L2 (24..64 equal, 192 no gain)
#endif
#ifndef SFFT_ROW_MINB
#define SFFT_ROW_MINB 3   // CTAs per SM the row kernels are compiled for
#endif
// v[e] = raw[e] * (x0^PW, x1^PW): x0 = xi(2j), x1 = xi(2j+1), j = tr + e*TPR; xi(2j) = xb + e*step
// (all values are multiples of 1/W, so the affine form is exact).
template <int EPT, int PW>
__device__ __forceinline__ void row_weight(const double2* raw, cplx* v, double xb, double step, double dx1) {
#pragma unroll
  for (int e = 0; e < EPT; ++e) {
    const double x0 = fma((double)e, step, xb), x1 = x0 + dx1;
    double w0 = x0, w1 = x1;
    if (PW >= 2) { w0 *= x0; w1 *= x1; }
    if (PW >= 3) { w0 *= x0; w1 *= x1; }
    v[e] = cmake(raw[e].x * w0, raw[e].y * w1);
  }
}

// hi[i] = sum_e v[e].x x0^(i+1) + v[e].y x1^(i+1), i < NDB (per-thread partial, sequential in e)
template <int EPT, int NDB>
__device__ __forceinline__ void row_extra_moments(const cplx* v, double xb, double step, double dx1, double* hi) {
#pragma unroll
  for (int i = 0; i < SFFT_MAX_DEG; ++i) hi[i] = 0.0;
#pragma unroll
  for (int e = 0; e < EPT; ++e) {
    const double x0 = fma((double)e, step, xb), x1 = x0 + dx1;
    double f0 = v[e].x, f1 = v[e].y;
#pragma unroll
    for (int i = 0; i < NDB; ++i) {
      f0 *= x0;
      f1 *= x1;
      hi[i] += f0 + f1;
    }
  }
}

// ------------------------------------------------------------------------------------------------
// Row pass of the fused build path: one CTA = one image (blockIdx.x % nimg, so the images of a pair run
// side by side and R stays in L2) of RB row PAIRS (2b, 2b+1), 2 RB TPR threads (256 at W = 4096), thread =
// (pair, row of the pair, tr).  The two rows of a pair are transformed side by side -- both go from global
// memory through the weighting into their first butterflies (registers only), the passes run on 2 RB
// sequences at once -- and leave the CTA together: the split step is shared, a thread takes half of its
// tr's bins for BOTH rows and writes, per column kx, the 32-byte pair {X_2b[kx], X_2b+1[kx]} into the
// row-group layout T[img][y/G][kx][y%G] (G = SFFT_T_G rows of one column are contiguous; kx in [0, NC]):
// whole 32-byte sectors, G/2 row pairs filling a 16 G-byte run that k_colb reads along y.  128 registers,
// two CTAs = 16 warps per SM (the kernel is latency-bound; a variant that transformed the two rows one
// after the other in 128-thread CTAs, the second row staged by cp.async, had 8-12 warps per SM and took
// 0.175 instead of 0.165 ms).  With colT = 0 the same kernel writes the row-major packed layout instead.
// A thread's EPT input elements j = tr + e*TPR are exactly the inputs of its first-pass butterfly; the
// mask is read once and kept as two bits per element.
// Fused reductions (moments != 0), all in a fixed order:
//   sum_x m xi^p R, p <= DK and sum_x m S : the DC bin of the image's own row transform;
//   sum_x m xi^a R, DK < a <= DK+DB and sum_x m xi^a S, 0 < a <= DB: DB extra sums on the
//     weighted values of the last R image and of the S image (shuffle tree, then warps in order);
//   sum_x m xi^a, a <= 2 DB: the closed-form whole-row sum minus the (rare) masked pixels.
__device__ __forceinline__ void row_st_pair(cplx* dst, cplx a, cplx b) {   // 32-byte streaming store
  asm volatile("st.global.cs.v4.f64 [%0], {%1, %2, %3, %4};\n" ::"l"(dst), "d"(a.x), "d"(a.y), "d"(b.x), "d"(b.y) : "memory");
}

template <int NC, int MINB>
__global__ void __launch_bounds__(256, MINB) k_row2_fwd(RowFwdParams P) {
  using C = FftCfg<NC>;
  constexpr int EPT = C::EPT;
  constexpr int TPR = NC / EPT;  // threads per row
  constexpr int LW = TPR < 32 ? TPR : 32;           // lanes of one row inside a warp
  constexpr int WPR = TPR / 32 > 0 ? TPR / 32 : 1;  // warps per row
  constexpr int NSLOT = 256 / LW;                   // (row, warp-of-row) slots of a CTA
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ double redM[ROW_NMA][NSLOT];
  __shared__ double redX[SFFT_MAX_DEG][NSLOT];
  cplx* s = reinterpret_cast<cplx*>(smem_raw);
  const int tid = threadIdx.x, nth = blockDim.x;
  const int nseq = nth / TPR;                       // rows of the CTA = 2 RB
  const int seq = tid / TPR, tr = tid - seq * TPR;
  const int pr = seq >> 1, rr = seq & 1;
  const int nimg = P.nR + P.withS;
  const int im = blockIdx.x % nimg;                 // images of one pair run side by side (R rows stay in L2)
  const int pairIdx = (blockIdx.x / nimg) * (nseq >> 1) + pr;
  const int y0 = 2 * pairIdx, y = y0 + rr;
  const int W = P.W, H = P.H;
  const double invW = 1.0 / (double)W;
  const double xb = (double)(4 * tr + 1 - W) * invW, step = (double)(4 * TPR) * invW, dx1 = 2.0 * invW;
  const int slot = tid / LW;
  const int pw = im < P.nR ? im : 0;
  const double* src = (im < P.nR ? P.R : P.S) + (size_t)y * W;

  double2 raw[EPT];
#pragma unroll
  for (int e = 0; e < EPT; ++e) raw[e] = ROW_LD(reinterpret_cast<const double2*>(src + 2 * (tr + e * TPR)));
  // the rows of a pair that starts about one wave of CTAs later are requested from L2 now (one request per
  // 128-byte line; R by the first image's CTA, S by the science image's, the mask with R)
  {
    const int pa = pairIdx + SFFT_ROW_AHEAD * (nseq >> 1);
    if (2 * pa + 1 < H && (im == 0 || im >= P.nR)) {
      const double* nb = (im < P.nR ? P.R : P.S) + (size_t)(2 * pa) * W;
      for (int l = tid; l < (2 * W) / 16; l += nth) asm volatile("prefetch.global.L2 [%0];" ::"l"(nb + 16 * l));
      if (im == 0 && P.mask)
        for (int l = tid; l < (2 * W) / 128; l += nth) asm volatile("prefetch.global.L2 [%0];" ::"l"(P.mask + (size_t)(2 * pa) * W + 128 * l));
    }
  }
  // mask bits: bit 2e = element 2j masked, bit 2e+1 = element 2j+1 masked, j = tr + e*TPR
  unsigned mbits = 0u;
  if (P.mask) {
    uchar2 mk[EPT];
#pragma unroll
    for (int e = 0; e < EPT; ++e) mk[e] = *reinterpret_cast<const uchar2*>(P.mask + (size_t)y * W + 2 * (tr + e * TPR));
#pragma unroll
    for (int e = 0; e < EPT; ++e) mbits |= (mk[e].x ? 1u : 0u) << (2 * e) | (mk[e].y ? 1u : 0u) << (2 * e + 1);
  }
  const bool momA = P.moments && im == 0;
  if (momA) {
    // masked part of sum_x m xi^a: only warps that hold a masked pixel do any work
    double ms[ROW_NMA];
#pragma unroll
    for (int a = 0; a < ROW_NMA; ++a) ms[a] = 0.0;
    if (__any_sync(0xffffffffu, mbits != 0u)) {
      unsigned mm = mbits;
      while (mm) {
        const int bit = __ffs(mm) - 1;
        mm &= mm - 1;
        const int j = tr + (bit >> 1) * TPR;
        const double x = (double)(4 * j + 1 + 2 * (bit & 1) - W) * invW;
        double pwr = 1.0;
#pragma unroll
        for (int a = 0; a < ROW_NMA; ++a) { ms[a] += pwr; pwr *= x; }
      }
#pragma unroll
      for (int a = 0; a < ROW_NMA; ++a) {
#pragma unroll
        for (int off = LW / 2; off > 0; off >>= 1) ms[a] += __shfl_xor_sync(0xffffffffu, ms[a], off);
      }
    }
    if ((tid & (LW - 1)) == 0) {
#pragma unroll
      for (int a = 0; a < ROW_NMA; ++a) redM[a][slot] = ms[a];
    }
  }
  if (mbits) {
#pragma unroll
    for (int e = 0; e < EPT; ++e) {
      if ((mbits >> (2 * e)) & 1u) raw[e].x = 0.0;
      if ((mbits >> (2 * e + 1)) & 1u) raw[e].y = 0.0;
    }
  }
  cplx v[EPT];
  switch (pw) {
    case 0:
#pragma unroll
      for (int e = 0; e < EPT; ++e) v[e] = raw[e];
      break;
    case 1: row_weight<EPT, 1>(raw, v, xb, step, dx1); break;
    case 2: row_weight<EPT, 2>(raw, v, xb, step, dx1); break;
    default: row_weight<EPT, 3>(raw, v, xb, step, dx1); break;
  }
  const bool extra = P.moments && P.DB > 0 && im >= P.nR - 1;
  if (extra) {
    double hi[SFFT_MAX_DEG];
    switch (P.DB) {
      case 1: row_extra_moments<EPT, 1>(v, xb, step, dx1, hi); break;
      case 2: row_extra_moments<EPT, 2>(v, xb, step, dx1, hi); break;
      default: row_extra_moments<EPT, 3>(v, xb, step, dx1, hi); break;
    }
#pragma unroll
    for (int i = 0; i < SFFT_MAX_DEG; ++i) {
#pragma unroll
      for (int off = LW / 2; off > 0; off >>= 1) hi[i] += __shfl_xor_sync(0xffffffffu, hi[i], off);
    }
    if ((tid & (LW - 1)) == 0) {
#pragma unroll
      for (int i = 0; i < SFFT_MAX_DEG; ++i) redX[i][slot] = hi[i];
    }
  }
  if constexpr (TPR >= 32 && 256 / TPR <= 8) {
    // a row's TPR threads (whole warps) exchange data only among themselves until the split: the passes meet
    // at a named barrier per row, so the rows of the CTA drift apart; one CTA barrier before the split
    fft_regs_to_smem<NC, -1, false>(v, s, tid, nth, nseq, P.twP, C::SEQ_STRIDE, FftSyncNamed<256 / TPR>{1 + seq, TPR});
    __syncthreads();
  } else {
    fft_regs_to_smem<NC, -1, false>(v, s, tid, nth, nseq, P.twP, C::SEQ_STRIDE);
  }

  // split of both rows of the pair; this thread: half rr of tr's bins
  const cplx* sA = s + (2 * pr) * C::SEQ_STRIDE;
  const cplx* sB = sA + C::SEQ_STRIDE;
  constexpr int G = SFFT_T_G;
  cplx* out = P.T + ((size_t)im * (H / G) + y0 / G) * (size_t)(NC + 1) * G + (y0 % G);   // column k at out + G k
  // row-major packed layout (generic build path, sfft_subtract): T[img][y][kx], kx < NC, column 0 = X[0] + i X[NC]
  cplx* outA = P.T + ((size_t)im * H + y0) * P.pitchT;
  cplx* outB = outA + P.pitchT;
  const bool grp = P.colT != 0;
  auto emit = [&](int k, cplx a, cplx b) {
    if (grp) row_st_pair(out + (size_t)G * k, a, b);
    else { ROW_ST(outA + k, a); ROW_ST(outB + k, b); }
  };
  constexpr int NIT = (NC / 2) / TPR, NH = NIT / 2;
  static_assert(NIT >= 2 && NIT % 2 == 0, "the split step is shared by the two rows' threads");
  const cplx tw0 = ldg2(P.twW + tr);
  cplx twrun = rr ? mul_split_root<EPT>(tw0, NH) : tw0;    // w^(tr + i TPR) = w^tr e^{-2 pi i i/(2 EPT)}
  cplx zk[2][NH], zm[2][NH];
#pragma unroll
  for (int i = 0; i < NH; ++i) {
    const int k = tr + (rr * NH + i) * TPR;
    const int pk = C::phys(k), pm = C::phys((NC - k) & (NC - 1));
    zk[0][i] = sA[pk]; zm[0][i] = cconj(sA[pm]);
    zk[1][i] = sB[pk]; zm[1][i] = cconj(sB[pm]);
  }
#pragma unroll
  for (int i = 0; i < NH; ++i) {
    const int k = tr + (rr * NH + i) * TPR;
    cplx xe[2], xo[2];
#pragma unroll
    for (int q = 0; q < 2; ++q) {
      xe[q] = cscale(cadd(zk[q][i], zm[q][i]), 0.5);
      xo[q] = cmul_mi(cscale(csub(zk[q][i], zm[q][i]), 0.5));
    }
    if (k == 0) {     // rr == 0, tr == 0, i == 0: DC and Nyquist bins, and the pair's moment writer
      double dc[2], ny[2];
#pragma unroll
      for (int q = 0; q < 2; ++q) { dc[q] = xe[q].x + xo[q].x; ny[q] = xe[q].x - xo[q].x; }
      if (grp) {
        emit(0, cmake(dc[0], 0.0), cmake(dc[1], 0.0));
        emit(NC, cmake(ny[0], 0.0), cmake(ny[1], 0.0));
      } else {
        emit(0, cmake(dc[0], ny[0]), cmake(dc[1], ny[1]));
      }
      if (P.moments) {
        for (int q = 0; q < 2; ++q) {
          const int yq = y0 + q, s0 = (2 * pr + q) * WPR;
          double* momS = P.rowMom + (size_t)P.nMomA * H + yq;
          double* momR = momS + (size_t)P.nMomS * H;
          if (im < P.nR) momR[(size_t)im * H] = dc[q]; else momS[0] = dc[q];
          if (extra) {
            double* dst = im < P.nR ? momR + (size_t)P.nR * H : momS + H;
            for (int ii = 0; ii < P.DB; ++ii) {
              double t = 0.0;
              for (int k2 = 0; k2 < WPR; ++k2) t += redX[ii][s0 + k2];
              dst[(size_t)ii * H] = t;
            }
          }
          if (momA) {
            for (int a = 0; a < P.nMomA; ++a) {
              double t = 0.0;
              for (int k2 = 0; k2 < WPR; ++k2) t += redM[a][s0 + k2];
              P.rowMom[(size_t)a * H + yq] = P.fullA[a] - t;
            }
          }
        }
      }
    } else {
      const cplx t0 = cmul(twrun, xo[0]), t1 = cmul(twrun, xo[1]);
      emit(k, cadd(xe[0], t0), cadd(xe[1], t1));
      emit(NC - k, cconj(csub(xe[0], t0)), cconj(csub(xe[1], t1)));
    }
    twrun = mul_split_root<EPT>(twrun, 1);
  }
  if (rr == 1 && tr == 0) {   // the middle bin k = NC/2 pairs with itself
    const cplx tw = ldg2(P.twW + NC / 2);
    cplx o[2];
#pragma unroll
    for (int q = 0; q < 2; ++q) {
      const cplx z = (q ? sB : sA)[C::phys(NC / 2)];
      const cplx zc = cconj(z);
      const cplx xe = cscale(cadd(z, zc), 0.5);
      const cplx xo = cmul_mi(cscale(csub(z, zc), 0.5));
      o[q] = cadd(xe, cmul(tw, xo));
    }
    emit(NC / 2, o[0], o[1]);
  }
}

// ------------------------------------------------------------------------------------------------

struct RowInvParams {
  const cplx* Mhat;  // [H][NC] packed row spectra of the model
  const double* S;
  const double* coeffs;  // device, length N; background part at offB
  double* D;
  int H, W, offB, DB;
  const cplx* twP;
  const cplx* twW;
};

// C2R row transform fused with D = S - M - B.  The merge (half spectrum -> packed complex
// sequence) is evaluated per element straight from global memory into the first butterfly, and
// the last pass leaves the row in registers for the subtraction, so shared memory carries only the
// exchanges between passes.
template <int NC, int MINB>
__global__ void __launch_bounds__(128, MINB) k_row_inv_sub(RowInvParams P) {
  using C = FftCfg<NC>;
  constexpr int EPT = C::EPT;
  constexpr int TPR = NC / EPT;
  constexpr int RL = fft_radix(NC, C::NPASS - 1);
  constexpr int NBL = NC / RL, ITL = EPT / RL;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx* s = reinterpret_cast<cplx*>(smem_raw);
  const int tid = threadIdx.x, nth = blockDim.x;
  const int RB = nth / TPR;
  const int r = tid / TPR, tr = tid - r * TPR;
  const int y0 = blockIdx.x * RB;
  const int W = P.W, H = P.H;
  const cplx* in = P.Mhat + (size_t)(y0 + r) * NC;
  // the science row is read only after the transform: ask L2 for it now (one request per 128-byte line)
  if ((tid & 7) == 0) {
#pragma unroll
    for (int m = 0; m < ITL; ++m) {
#pragma unroll
      for (int rr = 0; rr < RL; ++rr) {
        const double* a = P.S + (size_t)(y0 + r) * W + 2 * ((tid - r * TPR) + m * TPR + rr * NBL);
        asm volatile("prefetch.global.L2 [%0];" ::"l"(a));
      }
    }
  }
  // merge: Z[k] = Xe + i Xo,  Xe = (X[k] + conj(X[NC-k]))/2,  Xo = (X[k] - conj(X[NC-k]))/2 * e^{+2 pi i k/W}
  cplx v[EPT];
  {
    cplx xk[EPT], xm[EPT], tw[EPT];
    const cplx tw0 = ldg2(P.twW + tr);   // w^(tr + e TPR) = w^tr e^{-2 pi i e/(2 EPT)}: one table load, constant products
#pragma unroll
    for (int e = 0; e < EPT; ++e) {
      const int k = tr + e * TPR;
      xk[e] = in[k];
      xm[e] = in[(NC - k) & (NC - 1)];
    }
#pragma unroll
    for (int e = 0; e < EPT; ++e) tw[e] = e == 0 ? tw0 : mul_split_root<EPT>(tw0, e);
#pragma unroll
    for (int e = 0; e < EPT; ++e) {
      const int k = tr + e * TPR;
      if (k == 0) {
        v[e] = cmake(0.5 * (xk[e].x + xk[e].y), 0.5 * (xk[e].x - xk[e].y));  // (X[0], X[NC]) both real
      } else {
        const cplx m = cconj(xm[e]);
        const cplx xe = cscale(cadd(xk[e], m), 0.5);
        const cplx xo = cmul(cconj(tw[e]), cscale(csub(xk[e], m), 0.5));
        v[e] = cadd(xe, cmul_pi(xo));
      }
    }
  }
  fft_regs_to_regs<NC, +1, false>(v, s, tid, nth, RB, P.twP, C::SEQ_STRIDE);
  const double invW = 1.0 / (double)W, invNC = 1.0 / (double)NC;
#pragma unroll
  for (int m = 0; m < ITL; ++m) {
    int sq, j;
    fft_map<NBL, false, TPR>(tid, m, nth, RB, sq, j);
    const int y = y0 + sq;
    // background: B = sum_p cp[p] xi^p,  cp[p] = sum_q beta_(p,q) eta^q
    const double eta = (double)(2 * y + 1 - H) / (double)H;
    double cp[SFFT_MAX_DEG + 1];
#pragma unroll
    for (int p = 0; p <= SFFT_MAX_DEG; ++p) cp[p] = 0.0;
    for (int d = 0, t = 0; d <= P.DB; ++d)
      for (int q = 0; q <= d; ++q, ++t) {
        const double term = P.coeffs[P.offB + t] * ipow(eta, q);
#pragma unroll
        for (int p = 0; p <= SFFT_MAX_DEG; ++p)
          if (p == d - q) cp[p] += term;
      }
    const size_t rowoff = (size_t)y * W;
    double2 sv[RL];
#pragma unroll
    for (int rr = 0; rr < RL; ++rr) sv[rr] = *reinterpret_cast<const double2*>(P.S + rowoff + 2 * (j + rr * NBL));
#pragma unroll
    for (int rr = 0; rr < RL; ++rr) {
      const int n = j + rr * NBL;
      const cplx z = v[m * RL + rr];
      const double x0 = (double)(4 * n + 1 - W) * invW, x1 = (double)(4 * n + 3 - W) * invW;
      double b0 = cp[SFFT_MAX_DEG], b1 = cp[SFFT_MAX_DEG];
#pragma unroll
      for (int p = SFFT_MAX_DEG - 1; p >= 0; --p) {
        b0 = fma(b0, x0, cp[p]);
        b1 = fma(b1, x1, cp[p]);
      }
      double2 o;
      o.x = sv[rr].x - z.x * invNC - b0;
      o.y = sv[rr].y - z.y * invNC - b1;
      *reinterpret_cast<double2*>(P.D + rowoff + 2 * n) = o;
    }
  }
}

// ------------------------------------------------------------------------------------------------

static int row_threads(int NC, int H, int EPT) {
  const int TPR = NC / EPT;
  int RB = 128 / TPR;
  if (RB < 1) RB = 1;
  if (RB > H) RB = H;
  return RB * TPR;
}

template <int NC>
static sfft_status launch_row2_fwd_t(const RowFwdParams& P, cudaStream_t st) {
  using C = FftCfg<NC>;
  constexpr int TPR = NC / C::EPT;
  int RB = 128 / TPR;                               // row pairs per CTA
  if (RB < 1) RB = 1;
  if (RB > P.H / 2) RB = P.H / 2;
  const int nth = 2 * RB * TPR;
  const size_t smem = (size_t)2 * RB * C::SEQ_STRIDE * sizeof(cplx);
  constexpr int MINB = 2;
  SFFT_CUDA_TRY(cudaFuncSetAttribute(k_row2_fwd<NC, MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  k_row2_fwd<NC, MINB><<<(P.H / 2 / RB) * (P.nR + P.withS), nth, smem, st>>>(P);
  SFFT_LAUNCH_CHECK();
  return SFFT_OK;
}

template <int NC>
static sfft_status launch_row_inv_t(const RowInvParams& P, cudaStream_t st) {
  using C = FftCfg<NC>;
  const int nth = row_threads(NC, P.H, C::EPT);
  const int RB = nth / (NC / C::EPT);
  const size_t smem = (size_t)RB * C::SEQ_STRIDE * sizeof(cplx);
  constexpr int MINB = SFFT_ROW_MINB;
  SFFT_CUDA_TRY(cudaFuncSetAttribute(k_row_inv_sub<NC, MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  k_row_inv_sub<NC, MINB><<<P.H / RB, nth, smem, st>>>(P);
  SFFT_LAUNCH_CHECK();
  return SFFT_OK;
}

#define SFFT_DISPATCH_NC(NCV, CALL)                       \
  switch (NCV) {                                          \
    case 8: return CALL<8>(P, st);                        \
    case 16: return CALL<16>(P, st);                      \
    case 32: return CALL<32>(P, st);                      \
    case 64: return CALL<64>(P, st);                      \
    case 128: return CALL<128>(P, st);                    \
    case 256: return CALL<256>(P, st);                    \
    case 512: return CALL<512>(P, st);                    \
    case 1024: return CALL<1024>(P, st);                  \
    case 2048: return CALL<2048>(P, st);                  \
    default: return SFFT_ERR_UNSUPPORTED;                 \
  }

sfft_status sfft_launch_row_fwd(sfft_plan* p, const double* R, const double* S,
                                const unsigned char* mask, bool build, cplx* Tout, int pitchT, bool packed,
                                bool colT, cudaStream_t st, int* nl) {
  RowFwdParams P;
  P.R = R; P.S = S; P.mask = mask; P.H = p->H; P.W = p->W;
  P.nR = p->DK + 1; P.withS = (build && S) ? 1 : 0;   // S == NULL in a build: its row spectra are reused
  P.T = Tout; P.pitchT = pitchT; P.packed = packed ? 1 : 0; P.colT = colT ? 1 : 0; P.twP = p->twPNC; P.twW = p->twW;
  P.moments = build ? 1 : 0; P.DB = p->DB; P.nMomA = p->nMomA; P.nMomS = p->nMomS; P.nMomR = p->nMomR;
  P.rowMom = p->rowMom;
  for (int a = 0; a < ROW_NMA; ++a) P.fullA[a] = p->fullA[a];
  ++*nl;
  SFFT_DISPATCH_NC(p->NC, launch_row2_fwd_t)
}

sfft_status sfft_launch_row_inv_sub(sfft_plan* p, const double* S, const double* c, double* D,
                                    cudaStream_t st, int* nl) {
  RowInvParams P;
  P.Mhat = p->Mhat; P.S = S; P.coeffs = c; P.D = D; P.H = p->H; P.W = p->W;
  P.offB = p->L * p->TK; P.DB = p->DB; P.twP = p->twPNC; P.twW = p->twW;
  ++*nl;
  SFFT_DISPATCH_NC(p->NC, launch_row_inv_t)
}
