// Row-direction kernels.
//
//  k_row_fwd   : (a1)+(a2 first pass) -- generation of the polynomial-weighted, masked images
//                m xi^p R, m S, m xi^p fused into the first (row, R2C) pass of the 2-D FFT, plus
//                the fused fp64 reductions sum_x m xi^a and sum_x m xi^p S per row
//                (north_star subsystems (1),(2)).  The eta^q factor of a
//                monomial is a function of y only, so it commutes with the row transform and is
//                applied by the column pass: only DK+1 (not T_K) row transforms of R are needed.
//  k_row_inv_sub: (a6 last pass) -- C2R row transform of the mixed row spectra, fused with
//                D = S - M - B (north_star subsystem (6)).
//
// Real rows of length W are transformed as W/2-point complex FFTs of z[j] = x[2j] + i x[2j+1]
// with the standard split/merge post-(pre-)processing.  Output column 0 packs the two real
// bins: T[y][0] = X[0] + i X[W/2].
#include "fft_smem.cuh"

struct RowFwdParams {
  const double* R;
  const double* S;
  const unsigned char* mask;
  int H, W, nimg;
  RowImage img[8];
  cplx* T;  // [nimg][H][NC]
  const cplx* twNC;
  const cplx* twW;
  int moments, nMomA, nMomS;
  double* rowMom;  // [nMomA + nMomS][H]
};

template <int NC>
__global__ void __launch_bounds__(256) k_row_fwd(RowFwdParams P) {
  using C = FftCfg<NC>;
  constexpr int EPT = C::EPT;
  constexpr int TPR = NC / EPT;  // threads per row
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx* s = reinterpret_cast<cplx*>(smem_raw);
  const int tid = threadIdx.x, nth = blockDim.x;
  const int RB = nth / TPR;
  const int r = tid / TPR, tr = tid - r * TPR;
  const int y = blockIdx.x * RB + r;
  const int W = P.W, H = P.H;
  const double invW = 1.0 / (double)W;
  const size_t rowoff = (size_t)y * W;

  if (P.moments) {
    // fused reductions (tree order: per-thread partial -> binary tree over the row's threads)
    double acc[2 * SFFT_MAX_DEG + 1 + SFFT_MAX_DEG + 1];
    const int nq = P.nMomA + P.nMomS;
#pragma unroll
    for (int q = 0; q < 2 * SFFT_MAX_DEG + 2 + SFFT_MAX_DEG; ++q) acc[q] = 0.0;
    for (int e = 0; e < EPT; ++e) {
      const int j = tr + e * TPR;
      const double2 sv = *reinterpret_cast<const double2*>(P.S + rowoff + 2 * j);
      double m0 = 1.0, m1 = 1.0;
      if (P.mask) {
        const uchar2 mk = *reinterpret_cast<const uchar2*>(P.mask + rowoff + 2 * j);
        m0 = mk.x ? 0.0 : 1.0;
        m1 = mk.y ? 0.0 : 1.0;
      }
      const double x0 = (double)(4 * j + 1 - W) * invW, x1 = (double)(4 * j + 3 - W) * invW;
      double p0 = m0, p1 = m1;
      for (int a = 0; a < P.nMomA; ++a) {
        acc[a] += p0 + p1;
        if (a < P.nMomS) acc[P.nMomA + a] += p0 * sv.x + p1 * sv.y;
        p0 *= x0;
        p1 *= x1;
      }
    }
    double* red = reinterpret_cast<double*>(smem_raw);
    for (int q = 0; q < nq; ++q) red[q * nth + tid] = acc[q];
    __syncthreads();
    for (int off = TPR / 2; off > 0; off >>= 1) {
      if (tr < off)
        for (int q = 0; q < nq; ++q) red[q * nth + tid] += red[q * nth + tid + off];
      __syncthreads();
    }
    if (tr == 0)
      for (int q = 0; q < nq; ++q) P.rowMom[(size_t)q * H + y] = red[q * nth + tid];
    __syncthreads();
  }

  cplx* srow = s + r * C::SEQ_STRIDE;
  for (int im = 0; im < P.nimg; ++im) {
    const RowImage d = P.img[im];
    const double* src = d.src == 0 ? P.R : P.S;
#pragma unroll 4
    for (int e = 0; e < EPT; ++e) {
      const int j = tr + e * TPR;
      double2 v = make_double2(1.0, 1.0);
      if (d.src != 2) v = *reinterpret_cast<const double2*>(src + rowoff + 2 * j);
      if (d.masked && P.mask) {
        const uchar2 mk = *reinterpret_cast<const uchar2*>(P.mask + rowoff + 2 * j);
        if (mk.x) v.x = 0.0;
        if (mk.y) v.y = 0.0;
      }
      if (d.pxi > 0) {
        const double x0 = (double)(4 * j + 1 - W) * invW, x1 = (double)(4 * j + 3 - W) * invW;
        v.x *= ipow(x0, d.pxi);
        v.y *= ipow(x1, d.pxi);
      }
      srow[C::phys(j)] = v;
    }
    __syncthreads();
    fft_smem<NC, -1>(s, tid, nth, P.twNC);
    // split: X[k] = Xe + w^k Xo, X[NC-k] = conj(Xe - w^k Xo), w = e^{-2 pi i / W}
    cplx* out = P.T + ((size_t)im * H + y) * NC;
    for (int k = tr; k <= NC / 2; k += TPR) {
      const cplx zk = srow[C::phys(k)];
      const cplx zm = cconj(srow[C::phys((NC - k) & (NC - 1))]);
      const cplx xe = cscale(cadd(zk, zm), 0.5);
      const cplx xo = cmul_mi(cscale(csub(zk, zm), 0.5));
      if (k == 0) {
        out[0] = cmake(xe.x + xo.x, xe.x - xo.x);
      } else {
        const cplx t = cmul(ldg2(P.twW + k), xo);
        out[k] = cadd(xe, t);
        if (k != NC - k) out[NC - k] = cconj(csub(xe, t));
      }
    }
    __syncthreads();
  }
}

// ------------------------------------------------------------------------------------------------

struct RowInvParams {
  const cplx* Mhat;  // [H][NC] packed row spectra of the model
  const double* S;
  const double* coeffs;  // device, length N; background part at offB
  double* D;
  int H, W, offB, DB;
  const cplx* twNC;
  const cplx* twW;
};

template <int NC>
__global__ void __launch_bounds__(256) k_row_inv_sub(RowInvParams P) {
  using C = FftCfg<NC>;
  constexpr int EPT = C::EPT;
  constexpr int TPR = NC / EPT;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx* s = reinterpret_cast<cplx*>(smem_raw);
  const int tid = threadIdx.x, nth = blockDim.x;
  const int RB = nth / TPR;
  const int r = tid / TPR, tr = tid - r * TPR;
  const int y = blockIdx.x * RB + r;
  const int W = P.W, H = P.H;
  cplx* srow = s + r * C::SEQ_STRIDE;
  const cplx* in = P.Mhat + (size_t)y * NC;
  // merge: Z[k] = Xe + i Xo, Z[NC-k] = conj(Xe) + i conj(Xo),
  //        Xe = (X[k] + conj(X[NC-k]))/2, Xo = (X[k] - conj(X[NC-k]))/2 * e^{+2 pi i k/W}
  for (int k = tr; k <= NC / 2; k += TPR) {
    if (k == 0) {
      const cplx x0 = in[0];  // (X[0], X[NC]) both real
      srow[C::phys(0)] = cmake(0.5 * (x0.x + x0.y), 0.5 * (x0.x - x0.y));
    } else {
      const cplx xk = in[k];
      const cplx xm = cconj(in[NC - k]);
      const cplx xe = cscale(cadd(xk, xm), 0.5);
      const cplx xo = cmul(cconj(ldg2(P.twW + k)), cscale(csub(xk, xm), 0.5));
      srow[C::phys(k)] = cadd(xe, cmul_pi(xo));
      if (k != NC - k) srow[C::phys(NC - k)] = cadd(cconj(xe), cmul_pi(cconj(xo)));
    }
  }
  __syncthreads();
  fft_smem<NC, +1>(s, tid, nth, P.twNC);
  // background polynomial coefficients
  double beta[SFFT_MAX_T];
  int nb = 0;
  for (int d = 0; d <= P.DB; ++d)
    for (int q = 0; q <= d; ++q) { beta[nb] = P.coeffs[P.offB + nb]; ++nb; }
  const double invW = 1.0 / (double)W, invNC = 1.0 / (double)NC;
  const double eta = (double)(2 * y + 1 - H) / (double)H;
  const size_t rowoff = (size_t)y * W;
#pragma unroll 4
  for (int e = 0; e < EPT; ++e) {
    const int j = tr + e * TPR;
    const cplx z = srow[C::phys(j)];
    const double2 sv = *reinterpret_cast<const double2*>(P.S + rowoff + 2 * j);
    const double x0 = (double)(4 * j + 1 - W) * invW, x1 = (double)(4 * j + 3 - W) * invW;
    double b0 = 0.0, b1 = 0.0;
    int t = 0;
    for (int d = 0; d <= P.DB; ++d)
      for (int q = 0; q <= d; ++q) {
        const double eq = ipow(eta, q);
        b0 += beta[t] * ipow(x0, d - q) * eq;
        b1 += beta[t] * ipow(x1, d - q) * eq;
        ++t;
      }
    double2 o;
    o.x = sv.x - z.x * invNC - b0;
    o.y = sv.y - z.y * invNC - b1;
    *reinterpret_cast<double2*>(P.D + rowoff + 2 * j) = o;
  }
}

// ------------------------------------------------------------------------------------------------

static int rows_per_cta(int NC, int H) {
  const int EPT = (NC == 8 || NC == 32 || NC == 64 || NC == 512) ? 8 : 16;
  const int TPR = NC / EPT;
  int RB = 256 / TPR;
  if (RB < 1) RB = 1;
  if (NC >= 2048) RB = 2;
  if (RB > H) RB = H;
  return RB;
}

template <int NC>
static sfft_status launch_row_fwd_t(const RowFwdParams& P, cudaStream_t st) {
  using C = FftCfg<NC>;
  const int RB = rows_per_cta(NC, P.H);
  const int nth = RB * (NC / C::EPT);
  const size_t smem = (size_t)RB * C::SEQ_STRIDE * sizeof(cplx);
  SFFT_CUDA_TRY(cudaFuncSetAttribute(k_row_fwd<NC>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  k_row_fwd<NC><<<P.H / RB, nth, smem, st>>>(P);
  SFFT_LAUNCH_CHECK();
  return SFFT_OK;
}

template <int NC>
static sfft_status launch_row_inv_t(const RowInvParams& P, cudaStream_t st) {
  using C = FftCfg<NC>;
  const int RB = rows_per_cta(NC, P.H);
  const int nth = RB * (NC / C::EPT);
  const size_t smem = (size_t)RB * C::SEQ_STRIDE * sizeof(cplx);
  SFFT_CUDA_TRY(cudaFuncSetAttribute(k_row_inv_sub<NC>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  k_row_inv_sub<NC><<<P.H / RB, nth, smem, st>>>(P);
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
                                const unsigned char* mask, const RowImage* imgs, int nimg,
                                cplx* Tout, bool moments, cudaStream_t st, int* nl) {
  RowFwdParams P;
  P.R = R; P.S = S; P.mask = mask; P.H = p->H; P.W = p->W; P.nimg = nimg;
  for (int i = 0; i < nimg; ++i) P.img[i] = imgs[i];
  P.T = Tout; P.twNC = p->twNC; P.twW = p->twW;
  P.moments = moments ? 1 : 0; P.nMomA = p->nMomA; P.nMomS = p->nMomS; P.rowMom = p->rowMom;
  ++*nl;
  SFFT_DISPATCH_NC(p->NC, launch_row_fwd_t)
}

sfft_status sfft_launch_row_inv_sub(sfft_plan* p, const double* S, const double* c, double* D,
                                    cudaStream_t st, int* nl) {
  RowInvParams P;
  P.Mhat = p->Mhat; P.S = S; P.coeffs = c; P.D = D; P.H = p->H; P.W = p->W;
  P.offB = p->L * p->TK; P.DB = p->DB; P.twNC = p->twNC; P.twW = p->twW;
  ++*nl;
  SFFT_DISPATCH_NC(p->NC, launch_row_inv_t)
}
