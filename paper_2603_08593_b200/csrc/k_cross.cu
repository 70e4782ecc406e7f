// Fourier-domain cross products, lag-window inverse transforms and the gather into A, b
// (north_star subsystems (3),(4)).
//
// Only the (2D+1)^2 lags |dy|,|dx| <= D (D = 2w for kernel-kernel pairs, w otherwise) of each
// cross-correlation map C_{f,g} = irfft2(conj F_f . F_g) are ever read, so the inverse transform
// is evaluated only there:
//
//  k_cross<D>   : for every column kx, Y[dy][kx] = sum_ky conj(F_f) F_g e^{+2 pi i ky dy/H}, |dy|<=D.
//                 Output-pruned decimation: ky = b + (H/8) a, so
//                 Y[dy] = sum_b e^{2 pi i b dy/H} Z_b[dy mod 8],  Z_b = 8-point inverse DFT over a.
//                 One thread owns one (pair, column); a CTA owns 16 adjacent columns and a group of
//                 <= 21 pairs whose spectra tiles are staged once in shared memory (cp.async,
//                 double buffered); the 2D+1 accumulators live in registers.
//  k_lag_idft   : C[dy][dx] = (1/P) [ Re Y[dy][0] + (-1)^dx Re Y[dy][NC]
//                                     + 2 sum_{kx=1}^{NC-1} Re( Y[dy][kx] e^{2 pi i kx dx/W} ) ].
//  k_mom_final  : reduces the per-row moments of k_row2_fwd to sum m xi^a eta^b and sum m xi^p eta^q S.
//  k_gather     : A[tL+s, t'L+s'] = C_{t,t'}[(u-u', v-v')], b[tL+s] = C_{t,S}[(u,v)],
//                 A[tL+s, B t'] = C_{t,Psi t'}[(u,v)], A[B,B] and b_B from the moments.
#include "fft_smem.cuh"

struct CrossParams {
  const cplx* F;
  cplx* Y;
  const CrossGroup* groups;  // device array; blockIdx.y selects groups[g0 + blockIdx.y]
  int g0;
  int H, NC, pitch, nLag;
  int NB, log2NB;            // b values staged per pipeline stage (power of two, divides H/8)
  int c0;                    // windowed launches (half-ranges above 10): centre of the launch's 21 lags
  const cplx* twH;
};

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc) {
  const unsigned sa = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(sa), "l"(gsrc));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N)); }

// One CTA = SFFT_CR_CT adjacent columns x one group of <= SFFT_CR_GP pairs; thread = (pair, column).
// The group's spectra tiles are staged once in shared memory by cp.async (double buffered) and
// shared by all of its pairs, so every spectrum element leaves L2 once per group instead of once
// per pair.  Per staged b: x[a] = conj(F_f) F_g at ky = b + (H/8) a, 8-point inverse DFT over a,
// then the 2D+1 twiddled accumulations in registers.
// WIN (lag half-ranges above 10, i.e. w > 5): the launch computes the 2D+1 lags c0 - D .. c0 + D of a longer
// range, one twiddle load per lag (the symmetric pairing of +dy and -dy needs the window centred on 0).
template <int D, bool WIN = false>
__global__ void __launch_bounds__(SFFT_CR_GP * SFFT_CR_CT, 1) k_cross(CrossParams P) {
  constexpr int CT = SFFT_CR_CT;
  constexpr int NTH = SFFT_CR_GP * SFFT_CR_CT;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ CrossGroup G;
  const int tid = threadIdx.x;
  {
    const int* src = reinterpret_cast<const int*>(P.groups + P.g0 + blockIdx.y);
    int* dst = reinterpret_cast<int*>(&G);
    for (int e = tid; e < (int)(sizeof(CrossGroup) / sizeof(int)); e += NTH) dst[e] = src[e];
  }
  __syncthreads();
  const int ns = G.ns, NB = P.NB, lNB = P.log2NB;
  const int pl = tid / CT, col = tid - pl * CT;
  const bool has_pair = pl < G.np;
  const int la = has_pair ? G.la[pl] : 0, lb = has_pair ? G.lb[pl] : 0;
  const int kx0 = blockIdx.x * CT;
  const int N1 = P.H >> 3;
  const size_t specStride = (size_t)P.H * P.pitch;
  const int stageElems = ns * NB * 8 * CT;
  cplx* buf0 = reinterpret_cast<cplx*>(smem_raw);
  cplx* buf1 = buf0 + stageElems;

  auto issue = [&](int b0, cplx* buf) {
    for (int e = tid; e < stageElems; e += NTH) {
      const int c = e % CT, r = e / CT;            // r = (s*NB + bb)*8 + a
      const int a = r & 7, bb = (r >> 3) & (NB - 1), s = r >> (3 + lNB);
      const cplx* src = P.F + (size_t)G.spec[s] * specStride + (size_t)(b0 + bb + a * N1) * P.pitch + kx0 + c;
      cp_async16(buf + e, src);
    }
    cp_async_commit();
  };

  cplx acc[2 * D + 1];
#pragma unroll
  for (int i = 0; i < 2 * D + 1; ++i) acc[i] = cmake(0.0, 0.0);

  const int nst = N1 >> lNB;
  issue(0, buf0);
  for (int st = 0; st < nst; ++st) {
    cplx* cur = (st & 1) ? buf1 : buf0;
    if (st + 1 < nst) {
      issue((st + 1) << lNB, (st & 1) ? buf0 : buf1);
      cp_async_wait<1>();
    } else {
      cp_async_wait<0>();
    }
    __syncthreads();
    if (has_pair) {
      const cplx* pa = cur + (size_t)la * NB * 8 * CT + col;
      const cplx* pb = cur + (size_t)lb * NB * 8 * CT + col;
      for (int bb = 0; bb < NB; ++bb) {
        const int b = (st << lNB) + bb;
        cplx x[8];
#pragma unroll
        for (int a = 0; a < 8; ++a) x[a] = cmulc(pa[(bb * 8 + a) * CT], pb[(bb * 8 + a) * CT]);
        Dft<8, +1>::run(x);
        if constexpr (WIN) {
#pragma unroll
          for (int i = 0; i < 2 * D + 1; ++i) {
            const int dy = P.c0 + i - D;                         // (two's complement: & gives dy mod H)
            const cplx t = ldg2(P.twH + ((b * dy) & (P.H - 1)));  // e^{-2 pi i b dy/H}
            cfmac(acc[i], t, x[(i - D) & 7]);                    // += e^{+...} * Z[dy mod 8], c0 a multiple of 8
          }
        } else {
        acc[D] = cadd(acc[D], x[0]);
#pragma unroll
        for (int i = 1; i <= D; ++i) {
          const cplx t = ldg2(P.twH + ((b * i) & (P.H - 1)));  // e^{-2 pi i b i/H}
          cfmac(acc[D + i], t, x[i & 7]);                      // += e^{+...} * Z[i mod 8]
          cfma(acc[D - i], t, x[(8 - (i & 7)) & 7]);           // += e^{-...} * Z[-i mod 8]
        }
        }
      }
    }
    __syncthreads();
  }
  const int kx = kx0 + col;
  if (has_pair && kx <= P.NC) {
    const int Dp = G.D;  // the instantiated range may exceed the group's own half-range
    cplx* out = P.Y + ((size_t)G.pair[pl] * P.nLag) * P.pitch + kx;
#pragma unroll
    for (int i = 0; i < 2 * D + 1; ++i) {
      const int dy = (WIN ? P.c0 : 0) + i - D;
      if (dy >= -Dp && dy <= Dp) out[(size_t)(dy + Dp) * P.pitch] = acc[i];
    }
  }
}

template <int D>
static sfft_status launch_cross_t(const CrossParams& P, int ngroups, int maxns, cudaStream_t st) {
  const size_t smem = (size_t)2 * maxns * P.NB * 8 * SFFT_CR_CT * sizeof(cplx);
  SFFT_CUDA_TRY(cudaFuncSetAttribute(k_cross<D>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  dim3 grid(P.NC / SFFT_CR_CT + 1, ngroups);
  k_cross<D><<<grid, SFFT_CR_GP * SFFT_CR_CT, smem, st>>>(P);
  SFFT_LAUNCH_CHECK();
  return SFFT_OK;
}

// half-range Dfull > 10: 2 M + 1 launches of 25 lags each, centred on multiples of 24 (a multiple of 8, so the
// residue dy mod 8 of a lag is a compile-time constant in the unrolled loop)
#define SFFT_CR_WD 12
static sfft_status launch_cross_windows(int Dfull, CrossParams P, int ngroups, int maxns, cudaStream_t st, int* nl) {
  const size_t smem = (size_t)2 * maxns * P.NB * 8 * SFFT_CR_CT * sizeof(cplx);
  SFFT_CUDA_TRY(cudaFuncSetAttribute(k_cross<SFFT_CR_WD, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  dim3 grid(P.NC / SFFT_CR_CT + 1, ngroups);
  const int M = Dfull > SFFT_CR_WD ? (Dfull - SFFT_CR_WD + 2 * SFFT_CR_WD - 1) / (2 * SFFT_CR_WD) : 0;
  for (int m = -M; m <= M; ++m) {
    P.c0 = 2 * SFFT_CR_WD * m;
    k_cross<SFFT_CR_WD, true><<<grid, SFFT_CR_GP * SFFT_CR_CT, smem, st>>>(P);
    SFFT_LAUNCH_CHECK();
    if (m != -M) ++*nl;   // (the caller counts the first launch)
  }
  return SFFT_OK;
}

static sfft_status launch_cross_D(int D, const CrossParams& P, int ngroups, int maxns, cudaStream_t st, int* nl) {
  if (D > 10) return launch_cross_windows(D, P, ngroups, maxns, st, nl);
  switch (D) {
    case 0: case 1: return launch_cross_t<1>(P, ngroups, maxns, st);
    case 2: return launch_cross_t<2>(P, ngroups, maxns, st);
    case 3: return launch_cross_t<3>(P, ngroups, maxns, st);
    case 4: return launch_cross_t<4>(P, ngroups, maxns, st);
    case 5: return launch_cross_t<5>(P, ngroups, maxns, st);
    case 6: return launch_cross_t<6>(P, ngroups, maxns, st);
    case 7: case 8: return launch_cross_t<8>(P, ngroups, maxns, st);
    case 9: case 10: return launch_cross_t<10>(P, ngroups, maxns, st);
    default: return SFFT_ERR_UNSUPPORTED;
  }
}

sfft_status sfft_launch_cross(sfft_plan* p, cudaStream_t st, int* nl) {
  CrossParams P;
  P.F = p->F; P.Y = p->Y; P.groups = p->d_groups; P.H = p->H; P.NC = p->NC; P.pitch = p->pitch;
  P.nLag = p->nLag; P.twH = p->twH; P.c0 = 0;
  const int N1 = p->H / 8;
  auto pickNB = [&](int maxns) {  // largest staged depth whose double buffer fits in shared memory
    int nb = 4;
    while (nb > 1 && ((size_t)2 * maxns * nb * 8 * SFFT_CR_CT * sizeof(cplx) > 200 * 1024 || nb > N1)) nb >>= 1;
    return nb;
  };
  sfft_status s;
  // groups are sorted: kernel-kernel (D = 2w) first, then the D = w groups
  P.g0 = 0;
  P.NB = pickNB(p->maxnsKK); P.log2NB = P.NB == 4 ? 2 : (P.NB == 2 ? 1 : 0);
  ++*nl;
  { ProfScope ps(p, 2, st); s = launch_cross_D(2 * p->w, P, p->nGroupKK, p->maxnsKK, st, nl); }
  if (s != SFFT_OK) return s;
  P.g0 = p->nGroupKK;
  P.NB = pickNB(p->maxnsKO); P.log2NB = P.NB == 4 ? 2 : (P.NB == 2 ? 1 : 0);
  ++*nl;
  { ProfScope ps(p, 3, st); s = launch_cross_D(p->w, P, p->nGroupKO, p->maxnsKO, st, nl); }
  return s;
}

// ------------------------------------------------------------------------------------------------

struct LagParams {
  const cplx* Y;
  double* Cmap;  // [nPair][nLag][nLag]; pair with half-range D uses rows/cols [0, 2D]
  const PairDesc* pairs;
  int NC, W, pitch, nLag;
  int nPart;            // partial lag-row sets, added in order (1 on both build paths)
  size_t partStride;    // elements between two sets
  double invP;
  const cplx* twW;
};

#define LAG_TH 128   // 507 CTAs of 4 warps at Full: one wave (256 threads: 1.7 waves, and twice the reduction work per kx)
// LAG_MAXD = largest lag half-range of the instantiation: 10 (w <= 5) or 30 (w <= 15)

// One CTA per (pair, lag row): lanes run along kx (coalesced reads of the lag row), every thread
// keeps the 2D+1 partial sums of its kx values in registers, then a fixed-order reduction
// (warp shuffle tree, then the warps in order) so the result is reproducible.
template <int LAG_MAXD>
__global__ void __launch_bounds__(LAG_TH) k_lag_idft(LagParams P) {
  const int pair = blockIdx.x, dyi = blockIdx.y;
  const int D = P.pairs[pair].D;
  if (dyi > 2 * D) return;
  const int tid = threadIdx.x, lane = tid & 31, wrp = tid >> 5;
  const cplx* Yr = P.Y + ((size_t)pair * P.nLag + dyi) * P.pitch;
  double ap[LAG_MAXD + 1], am[LAG_MAXD + 1];
#pragma unroll
  for (int dx = 0; dx <= LAG_MAXD; ++dx) { ap[dx] = 0.0; am[dx] = 0.0; }
  // four kx per step: their class partials and first twiddles are requested together; the twiddles
  // of the higher lags follow by the recurrence t_dx = t_{dx-1} t_1 (<= 10 products, error ~1e-15)
  for (int kx0 = 1 + tid; kx0 < P.NC; kx0 += 4 * LAG_TH) {
    cplx ys[4], t1[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int kx = kx0 + u * LAG_TH;
      const bool in = kx < P.NC;
      ys[u] = in ? Yr[kx] : cmake(0.0, 0.0);
      t1[u] = in ? ldg2(P.twW + kx) : cmake(1.0, 0.0);   // (c, -s) of angle 2 pi kx / W
    }
    for (int q = 1; q < P.nPart; ++q) {
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int kx = kx0 + u * LAG_TH;
        if (kx < P.NC) ys[u] = cadd(ys[u], Yr[kx + q * P.partStride]);
      }
    }
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const cplx y = ys[u];
      ap[0] += y.x;
      cplx t = t1[u];
#pragma unroll
      for (int dx = 1; dx <= LAG_MAXD; ++dx) {
        if (dx <= D) {
          ap[dx] = fma(y.x, t.x, ap[dx]);   // sum Re y cos(dx th)
          am[dx] = fma(y.y, t.y, am[dx]);   // -sum Im y sin(dx th);  Re(y e^{+-i dx th}) = their sum / difference
          t = cmul(t, t1[u]);
        }
      }
    }
  }
  __shared__ double red[2][LAG_MAXD + 1][LAG_TH / 32];
#pragma unroll
  for (int dx = 0; dx <= LAG_MAXD; ++dx) {
    double a = ap[dx] + am[dx], b = ap[dx] - am[dx];
    if (dx == 0) { a = ap[0]; b = ap[0]; }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
      a += __shfl_xor_sync(0xffffffffu, a, off);
      b += __shfl_xor_sync(0xffffffffu, b, off);
    }
    if (lane == 0) { red[0][dx][wrp] = a; red[1][dx][wrp] = b; }
  }
  __syncthreads();
  if (tid <= D) {
    const int dx = tid;
    double sp = 0.0, sm = 0.0;
    for (int k = 0; k < LAG_TH / 32; ++k) { sp += red[0][dx][k]; sm += red[1][dx][k]; }
    if (dx == 0) sm = sp;
    double y0 = Yr[0].x, yn = Yr[P.NC].x;
    for (int q = 1; q < P.nPart; ++q) { y0 += Yr[q * P.partStride].x; yn += Yr[P.NC + q * P.partStride].x; }
    const double sgn = (dx & 1) ? -1.0 : 1.0;
    double* out = P.Cmap + ((size_t)pair * P.nLag + dyi) * P.nLag;
    out[D + dx] = (y0 + sgn * yn + 2.0 * sp) * P.invP;
    out[D - dx] = (y0 + sgn * yn + 2.0 * sm) * P.invP;
  }
}

struct MomParams {
  const double* rowMom;  // [nMomA + nMomS + nMomR][H]
  double* mom;           // [nMomA*nMomA] then [TB] then [nMomR*nMomR]
  int H, nMomA, nMomS, nMomR, TB;
  int monoB[SFFT_MAX_T][2];
};

__global__ void __launch_bounds__(256) k_mom_final(MomParams P) {
  // block q < nMomA^2: (a,b) = (q / nMomA, q % nMomA) -> sum_y eta^b rowMom[a][y]
  // next TB blocks: background rhs t' -> sum_y eta^q rowMomS[p][y]; then nMomR^2 blocks: mu_ab
  const int q = blockIdx.x;
  int row, pw;
  if (q < P.nMomA * P.nMomA) {
    row = q / P.nMomA;
    pw = q % P.nMomA;
  } else if (q < P.nMomA * P.nMomA + P.TB) {
    const int t = q - P.nMomA * P.nMomA;
    row = P.nMomA + P.monoB[t][0];
    pw = P.monoB[t][1];
  } else {   // mu_ab = sum m R xi^a eta^b
    const int e = q - P.nMomA * P.nMomA - P.TB;
    row = P.nMomA + P.nMomS + e / P.nMomR;
    pw = e % P.nMomR;
  }
  const double* src = P.rowMom + (size_t)row * P.H;
  const double invH = 1.0 / (double)P.H;
  double acc = 0.0;
  for (int y = threadIdx.x; y < P.H; y += 256)
    acc += ipow((double)(2 * y + 1 - P.H) * invH, pw) * src[y];
  __shared__ double red[256];
  red[threadIdx.x] = acc;
  __syncthreads();
  for (int off = 128; off > 0; off >>= 1) {
    if (threadIdx.x < off) red[threadIdx.x] += red[threadIdx.x + off];
    __syncthreads();
  }
  if (threadIdx.x == 0) P.mom[q] = red[0];
}

struct GatherParams {
  const double* Cmap;
  const double* mom;
  const double* kbCorr;   // [(t*L + s)*TB + t'] sparse part of the kernel-background block (k_kb.cu)
  const double* kbStrip;  // [(t*L + s)*TB + t'] part of the fully masked target rows (k_kb_strip)
  double* A;
  double* b;
  int w, L, TK, TB, N, nLag, nMomA, nMomR, H, W;
  int monoK[SFFT_MAX_T][2], monoB[SFFT_MAX_T][2];
};

__device__ __forceinline__ double binom(int n, int k) {
  double r = 1.0;
  for (int i = 1; i <= k; ++i) r = r * (double)(n - k + i) / (double)i;
  return r;
}

__global__ void __launch_bounds__(256) k_gather(GatherParams P) {
  const int N = P.N, L = P.L, w = P.w, S1 = 2 * w + 1;
  const int nK = L * P.TK;
  const int nKK = P.TK * (P.TK + 1) / 2;
  const size_t lag2 = (size_t)P.nLag * P.nLag;
  // grid: y = row of A (y = N: the right-hand side), x = blocks of 256 columns -- 32-bit index arithmetic only
  const int row = blockIdx.y, col = blockIdx.x * 256 + threadIdx.x;
  if (col >= N) return;
  {
    if (row == N) {  // right-hand side
      const int i = col;
      double v;
      if (i < nK) {
        const int t = i / L, s = i - t * L;
        const int u = s % S1 - w, vv = s / S1 - w;
        const int pair = nKK + t;  // (t, S)
        v = P.Cmap[pair * lag2 + (size_t)(vv + w) * P.nLag + (u + w)];
      } else {
        v = P.mom[P.nMomA * P.nMomA + (i - nK)];
      }
      P.b[i] = v;
      return;
    }
    const int i = row, j = col;
    double v;
    if (i < nK && j < nK) {
      int t = i / L, s = i - t * L, t2 = j / L, s2 = j - t2 * L;
      int du = (s % S1) - (s2 % S1), dv = (s / S1) - (s2 / S1);
      if (t > t2) { int tmp = t; t = t2; t2 = tmp; du = -du; dv = -dv; }
      // auto-correlation maps are even: read one canonical half so A is bitwise symmetric
      if (t == t2 && (dv < 0 || (dv == 0 && du < 0))) { du = -du; dv = -dv; }
      // pair index of (t,t2), t <= t2, in row-major upper-triangular order
      const int pair = t * P.TK - t * (t - 1) / 2 + (t2 - t);
      const int D = 2 * w;
      v = P.Cmap[pair * lag2 + (size_t)(dv + D) * P.nLag + (du + D)];
    } else if (i < nK || j < nK) {
      const int ik = i < nK ? i : j, ib = (i < nK ? j : i) - nK;
      const int t = ik / L, s = ik - t * L;
      const int u = s % S1 - w, vv = s / S1 - w;
      // moments part: sum_x' R~_t(x') P_t'(x' + (u,v)), the polynomial expanded about x'
      const int pk = P.monoK[t][0], qk = P.monoK[t][1], pb = P.monoB[ib][0], qb = P.monoB[ib][1];
      const double dx = 2.0 * (double)u / (double)P.W, dy = 2.0 * (double)vv / (double)P.H;
      const double* mu = P.mom + P.nMomA * P.nMomA + P.TB;
      double acc = 0.0;
      for (int ii = 0; ii <= pb; ++ii) {
        const double cx = binom(pb, ii) * ipow(dx, pb - ii);
        for (int jj = 0; jj <= qb; ++jj)
          acc += cx * binom(qb, jj) * ipow(dy, qb - jj) * mu[(pk + ii) * P.nMomR + (qk + jj)];
      }
      v = acc - P.kbStrip[((size_t)t * L + s) * P.TB + ib] + P.kbCorr[((size_t)t * L + s) * P.TB + ib];
    } else {
      const int a = i - nK, c = j - nK;
      const int pa = P.monoB[a][0] + P.monoB[c][0], qa = P.monoB[a][1] + P.monoB[c][1];
      v = P.mom[pa * P.nMomA + qa];
    }
    P.A[(size_t)i * N + j] = v;
  }
}

struct StripParams {
  const int* fmList;      // fully masked target rows: count, then the rows in ascending order
  const double* rowMomR;  // [nMomR][H] sum_x m R xi^a per row
  double* kbStrip;        // [(t*L + s)*TB + t']
  int w, L, TK, TB, H, W;
  int monoK[SFFT_MAX_T][2], monoB[SFFT_MAX_T][2];
};

// Part of the kernel-background block that belongs to fully masked target rows y (k_kb.cu):
//   sum_y eta'^qk (eta' + dy)^qb sum_ii C(pb,ii) dx^(pb-ii) rowMomR[pk+ii][y'],  y' = wrap(y - v) the source
// row and eta' its own coordinate; one thread per entry, rows in ascending order.
__global__ void __launch_bounds__(128) k_kb_strip(StripParams P) {
  const int e = blockIdx.x * 128 + threadIdx.x;
  if (e >= P.TK * P.L * P.TB) return;
  const int ib = e % P.TB, ik = e / P.TB, t = ik / P.L, s = ik - t * P.L, S1 = 2 * P.w + 1;
  const int u = s % S1 - P.w, vv = s / S1 - P.w;
  const int pk = P.monoK[t][0], qk = P.monoK[t][1], pb = P.monoB[ib][0], qb = P.monoB[ib][1];
  const double dx = 2.0 * (double)u / (double)P.W, dy = 2.0 * (double)vv / (double)P.H;
  double cx[SFFT_MAX_DEG + 1];
  for (int ii = 0; ii <= pb; ++ii) cx[ii] = binom(pb, ii) * ipow(dx, pb - ii);
  double strip = 0.0;
  const int nfm = P.fmList[0];
  for (int f = 0; f < nfm; ++f) {
    const int ys = (P.fmList[1 + f] - vv + P.H) & (P.H - 1);
    const double etas = (double)(2 * ys + 1 - P.H) / (double)P.H;
    double rsum = 0.0;
    for (int ii = 0; ii <= pb; ++ii) rsum += cx[ii] * P.rowMomR[(size_t)(pk + ii) * P.H + ys];
    strip += ipow(etas, qk) * ipow(etas + dy, qb) * rsum;
  }
  P.kbStrip[e] = strip;
}

// final reduction of the row moments (depends on the row pass only)
sfft_status sfft_launch_moments(sfft_plan* p, cudaStream_t st, int* nl) {
  MomParams MP;
  MP.rowMom = p->rowMom; MP.mom = p->mom; MP.H = p->H; MP.nMomA = p->nMomA; MP.nMomS = p->nMomS; MP.nMomR = p->nMomR;
  MP.TB = p->TB;
  for (int t = 0; t < p->TB; ++t) { MP.monoB[t][0] = p->monoB[t][0]; MP.monoB[t][1] = p->monoB[t][1]; }
  k_mom_final<<<p->nMomA * p->nMomA + p->TB + p->nMomR * p->nMomR, 256, 0, st>>>(MP);
  SFFT_LAUNCH_CHECK();
  ++*nl;
  StripParams SP;
  SP.fmList = p->fmList; SP.rowMomR = p->rowMom + (size_t)(p->nMomA + p->nMomS) * p->H; SP.kbStrip = p->kbStrip;
  SP.w = p->w; SP.L = p->L; SP.TK = p->TK; SP.TB = p->TB; SP.H = p->H; SP.W = p->W;
  for (int t = 0; t < p->TB; ++t) { SP.monoB[t][0] = p->monoB[t][0]; SP.monoB[t][1] = p->monoB[t][1]; }
  for (int t = 0; t < p->TK; ++t) { SP.monoK[t][0] = p->monoK[t][0]; SP.monoK[t][1] = p->monoK[t][1]; }
  k_kb_strip<<<(p->TK * p->L * p->TB + 127) / 128, 128, 0, st>>>(SP);
  SFFT_LAUNCH_CHECK();
  ++*nl;
  return SFFT_OK;
}

sfft_status sfft_launch_lag_gather(sfft_plan* p, double* A, double* b, cudaStream_t st, int* nl) {
  LagParams LP;
  LP.Y = p->Y; LP.Cmap = p->Cmap; LP.pairs = p->d_pairs; LP.NC = p->NC; LP.W = p->W;
  LP.pitch = p->pitch; LP.nLag = p->nLag; LP.invP = 1.0 / ((double)p->H * (double)p->W);
  LP.twW = p->twW;
  LP.nPart = p->nPart; LP.partStride = (size_t)p->nPair * p->nLag * p->pitch;
  dim3 g1(p->nPair, p->nLag);
  if (p->Dmax <= 10) k_lag_idft<10><<<g1, LAG_TH, 0, st>>>(LP);
  else k_lag_idft<30><<<g1, LAG_TH, 0, st>>>(LP);
  SFFT_LAUNCH_CHECK();
  ++*nl;
  GatherParams GP;
  GP.Cmap = p->Cmap; GP.mom = p->mom; GP.A = A; GP.b = b; GP.w = p->w; GP.L = p->L; GP.TK = p->TK;
  GP.TB = p->TB; GP.N = p->N; GP.nLag = p->nLag; GP.nMomA = p->nMomA; GP.nMomR = p->nMomR;
  GP.H = p->H; GP.W = p->W; GP.kbCorr = p->kbCorr;
  GP.kbStrip = p->kbStrip;
  for (int t = 0; t < p->TB; ++t) { GP.monoB[t][0] = p->monoB[t][0]; GP.monoB[t][1] = p->monoB[t][1]; }
  for (int t = 0; t < p->TK; ++t) { GP.monoK[t][0] = p->monoK[t][0]; GP.monoK[t][1] = p->monoK[t][1]; }
  const dim3 blocks((p->N + 255) / 256, p->N + 1);   // y = row of A, y = N: the right-hand side
  k_gather<<<blocks, 256, 0, st>>>(GP);
  SFFT_LAUNCH_CHECK();
  ++*nl;
  return SFFT_OK;
}
