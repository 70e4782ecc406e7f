// Kernel-background cross block of the normal matrix without any transform
// (north_star subsystems (1),(4); SURVEY.md §8(d) "lean" plan).
//
//   A[(s,t),t'] = sum_x R~_t(x - u) Psi_t'(x),   R~_t = m P_t R,  Psi_t' = m P_t',  s <-> u = (u,v),
// indices mod (W,H).  With x' = x - u and the polynomial continued beyond the edges,
//
//   A[(s,t),t'] = sum_x' R~_t(x') P_t'(x' + u)                                        (I)
//               + sum_{x special} R~_t(wrap(x - u)) [ m(x) P_t'(x) - P_t'(wrap(x - u) + u) ]   (II)
//
// where a target pixel x is "special" when it is masked or lies within w of an edge (only those
// can be masked or be reached by a wrapped shift); for an unmasked target reached without
// wrapping the bracket vanishes identically.  (I) is a combination of the moments
// mu_ab = sum m R xi^a eta^b, a+b <= DK+DB (fused into the row pass, k_rows.cu), expanded in
// k_gather with delta_x = 2u/W, delta_y = 2v/H; (II) is the sparse sum evaluated here.
// Fully masked target rows (a CCD's top and bottom border) are taken out of the sparse sum: all W
// targets of such a row y are masked, so their part of (II) is -sum_x' R~_t(x', y') P_t'(x'+u, y'+v)
// over the WHOLE source row y' = wrap(y - v), a combination of the row moments sum_x m R xi^a that
// the row pass already delivers (evaluated in k_gather).
// Every sum has a fixed order (per-row ordered compaction, per-thread sequential partials, ordered
// final reduction), so the block is reproducible run to run.
#include "sfft_common.cuh"

#define KB_TH 128
#ifndef KB_CH
#define KB_CH 128   // special pixels staged per chunk
#endif

// Monomial t of the order "for d: for q <= d: p = d - q" as compile-time functions, so that the
// unrolled loops below multiply by register-held powers without any table lookups.
__host__ __device__ constexpr int mono_d(int t) { int d = 0; while ((d + 1) * (d + 2) / 2 <= t) ++d; return d; }
__host__ __device__ constexpr int mono_q(int t) { return t - mono_d(t) * (mono_d(t) + 1) / 2; }
__host__ __device__ constexpr int mono_p(int t) { return mono_d(t) - mono_q(t); }

__device__ __forceinline__ void powers(double x, double* pw) {   // pw[k] = x^k, k <= SFFT_MAX_DEG
  pw[0] = 1.0;
#pragma unroll
  for (int k = 1; k <= SFFT_MAX_DEG; ++k) pw[k] = pw[k - 1] * x;
}

__device__ __forceinline__ bool sp_strip(int x, int y, int W, int H, int w) {
  return x < w || x >= W - w || y < w || y >= H - w;
}

// One warp per row, 16 pixels per lane and step.  FILL = false: count the row's special pixels.
// FILL = true: write them, in x order, at spOff[y].
// A row whose W pixels are all masked is not listed: its whole contribution is a combination of
// the source rows' moments (k_gather), see the header of this file; fmFlag[y] marks such rows.
template <bool FILL>
__global__ void __launch_bounds__(256) k_sp_rows(const unsigned char* __restrict__ mask, int H, int W, int w,
                                                 int* spCount, const int* __restrict__ spOff, int* spList,
                                                 int* fmFlag) {
  const int lane = threadIdx.x & 31;
  const int y = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (y >= H) return;
  if (FILL && fmFlag[y]) return;
  const int base = FILL ? spOff[y] : 0;
  int nmasked = 0;
  const bool edge_row = y < w || y >= H - w;
  int total = 0;
  for (int k = 0; k < (W + 511) / 512; ++k) {   // uniform trip count for the shuffles
    const int x0 = k * 512 + lane * 16;
    unsigned flags = 0u, mk = 0u;
    if (x0 < W) {   // W is a multiple of 32, so a lane's 16 pixels are all inside or all outside
      if (mask) {
        const uint4 m16 = *reinterpret_cast<const uint4*>(mask + (size_t)y * W + x0);
        const unsigned wd[4] = {m16.x, m16.y, m16.z, m16.w};
#pragma unroll
        for (int q = 0; q < 4; ++q)
#pragma unroll
          for (int i = 0; i < 4; ++i)
            if ((wd[q] >> (8 * i)) & 0xffu) mk |= 1u << (4 * q + i);
      }
      flags = mk;
      nmasked += __popc(mk);
      if (edge_row) flags = 0xffffu;
      else if (x0 < w || x0 + 16 > W - w) {
#pragma unroll
        for (int i = 0; i < 16; ++i)
          if (x0 + i < w || x0 + i >= W - w) flags |= 1u << i;
      }
    }
    const int c = __popc(flags);
    if (FILL) {
      int incl = c;
#pragma unroll
      for (int off = 1; off < 32; off <<= 1) {
        const int t = __shfl_up_sync(0xffffffffu, incl, off);
        if (lane >= off) incl += t;
      }
      int pos = base + total + incl - c;
      while (flags) {
        const int i = __ffs(flags) - 1;
        flags &= flags - 1;
        spList[pos++] = (y * W + x0 + i) | (((mk >> i) & 1u) ? (int)0x80000000u : 0);
      }
      total += __shfl_sync(0xffffffffu, incl, 31);
    } else {
      total += c;
    }
  }
  if (!FILL) {
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
      total += __shfl_xor_sync(0xffffffffu, total, off);
      nmasked += __shfl_xor_sync(0xffffffffu, nmasked, off);
    }
    if (lane == 0) {
      const int full = nmasked == W;
      fmFlag[y] = full;
      spCount[y] = full ? 0 : total;
    }
  }
}

// Exclusive scan of the per-row counts (H <= 4096) by one CTA.
// Also compacts the fully masked rows, in ascending order, into fmList[1..], fmList[0] = their number.
__global__ void __launch_bounds__(1024) k_sp_scan(const int* __restrict__ spCount, int* spOff, int H,
                                                  const int* __restrict__ fmFlag, int* fmList) {
  __shared__ int part[1024];
  const int tid = threadIdx.x;
  const int per = (H + 1023) / 1024;
  int loc[4] = {0, 0, 0, 0};
  int sum = 0;
  {
    int fl[4] = {0, 0, 0, 0}, fsum = 0;
    for (int i = 0; i < per; ++i) {
      const int y = tid * per + i;
      fl[i] = y < H ? fmFlag[y] : 0;
      fsum += fl[i];
    }
    part[tid] = fsum;
    __syncthreads();
    for (int off = 1; off < 1024; off <<= 1) {
      const int t = tid >= off ? part[tid - off] : 0;
      __syncthreads();
      part[tid] += t;
      __syncthreads();
    }
    int run = part[tid] - fsum;
    for (int i = 0; i < per; ++i)
      if (fl[i]) fmList[1 + run++] = tid * per + i;
    if (tid == 1023) fmList[0] = part[1023];
    __syncthreads();
  }
  for (int i = 0; i < per; ++i) {
    const int y = tid * per + i;
    loc[i] = y < H ? spCount[y] : 0;
    sum += loc[i];
  }
  part[tid] = sum;
  __syncthreads();
  for (int off = 1; off < 1024; off <<= 1) {
    const int t = tid >= off ? part[tid - off] : 0;
    __syncthreads();
    part[tid] += t;
    __syncthreads();
  }
  int run = part[tid] - sum;
  for (int i = 0; i < per; ++i) {
    const int y = tid * per + i;
    if (y < H) spOff[y] = run;
    run += loc[i];
  }
  if (tid == 1023) spOff[H] = part[1023];
}

struct KbParams {
  const double* R;
  const unsigned char* mask;
  const int* spOff;
  const int* spList;
  double* part;   // [gridDim.x * nsub][TK][L][TB]
  int H, W, w, L, TK, TB, nsub;
  int monoK[SFFT_MAX_T][2], monoB[SFFT_MAX_T][2];
};

// grid = (SFFT_KB_NBLK, TK/NT); thread = (shift s, pixel subset sub).  Each thread walks its share
// of the special pixels sequentially and keeps the NT x TB partial sums of its rows (s, t),
// t = blockIdx.y*NT .. +NT-1, in registers, so the index arithmetic and the two scattered source
// loads of a (pixel, shift) are shared by all its monomial pairs.
template <int NT, int TB, int T0>
__device__ __forceinline__ void kb_corr_body(const KbParams& P) {
  __shared__ int sx[KB_CH], sy[KB_CH];
  __shared__ double sP[KB_CH][TB];   // P_t'(x) of the staged targets
  __shared__ unsigned char sm[KB_CH];
  const int tid = threadIdx.x;
  const int W = P.W, H = P.H, w = P.w, S1 = 2 * w + 1;
  // L <= KB_TH: thread = (shift s, pixel subset sub), grid.z = 1; L > KB_TH (w > 5): one shift per thread, the
  // shifts spread over grid.z CTAs, a single subset
  const bool wide = P.L > KB_TH;
  const int s = wide ? (int)blockIdx.z * KB_TH + tid : tid % P.L, sub = wide ? 0 : tid / P.L;
  const bool active = wide ? s < P.L : sub < P.nsub;
  const int u = s % S1 - w, v = s / S1 - w;
  const double invW = 1.0 / (double)W, invH = 1.0 / (double)H;
  const int nsp = P.spOff[H];
  double acc[NT][TB];
#pragma unroll
  for (int a = 0; a < NT; ++a)
#pragma unroll
    for (int i = 0; i < TB; ++i) acc[a][i] = 0.0;
  for (int c0 = blockIdx.x * KB_CH; c0 < nsp; c0 += gridDim.x * KB_CH) {
    const int n = min(KB_CH, nsp - c0);
    __syncthreads();
    if (tid < n) {
      const int e = P.spList[c0 + tid];
      const int pix = e & 0x7fffffff;
      const int y = pix / W, x = pix - y * W;
      sx[tid] = x; sy[tid] = y; sm[tid] = e < 0 ? 1 : 0;
      const double xi = (double)(2 * x + 1 - W) * invW, eta = (double)(2 * y + 1 - H) * invH;
      double xp[SFFT_MAX_DEG + 1], ep[SFFT_MAX_DEG + 1];
      powers(xi, xp);
      powers(eta, ep);
#pragma unroll
      for (int tb = 0; tb < TB; ++tb) sP[tid][tb] = xp[mono_p(tb)] * ep[mono_q(tb)];
    }
    __syncthreads();
    if (!active) continue;
    // four pixels per step, their source loads (mask byte, R value) issued together: the loop is
    // bound by the latency of these scattered loads
    for (int i0 = sub; i0 < n; i0 += 4 * P.nsub) {
      int xw[4], yw[4];
      bool use[4], wrapped[4], masked[4];
      unsigned char ms[4];
      double rv[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const int i = i0 + k * P.nsub;
        use[k] = i < n;
        const int x = use[k] ? sx[i] : 0, y = use[k] ? sy[i] : 0;
        masked[k] = use[k] && sm[i] != 0;
        const int xs = x - u, ys = y - v;
        wrapped[k] = xs < 0 || xs >= W || ys < 0 || ys >= H;
        use[k] = use[k] && (wrapped[k] || masked[k]);
        xw[k] = xs & (W - 1);
        yw[k] = ys & (H - 1);
      }
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const size_t so = (size_t)yw[k] * W + xw[k];
        ms[k] = (use[k] && P.mask) ? P.mask[so] : 0;
        rv[k] = use[k] ? P.R[so] : 0.0;
      }
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        if (!use[k] || ms[k]) continue;   // R~ vanishes at a masked source
        const int i = i0 + k * P.nsub;
        const double xis = (double)(2 * xw[k] + 1 - W) * invW, etas = (double)(2 * yw[k] + 1 - H) * invH;
        double q[TB];
        if (!wrapped[k]) {
#pragma unroll
          for (int tb = 0; tb < TB; ++tb) q[tb] = -sP[i][tb];
        } else {
          // unwrapped target coordinates: source + shift
          const double xit = (double)(2 * (xw[k] + u) + 1 - W) * invW, etat = (double)(2 * (yw[k] + v) + 1 - H) * invH;
          double xp[SFFT_MAX_DEG + 1], ep[SFFT_MAX_DEG + 1];
          powers(xit, xp);
          powers(etat, ep);
#pragma unroll
          for (int tb = 0; tb < TB; ++tb)
            q[tb] = (masked[k] ? 0.0 : sP[i][tb]) - xp[mono_p(tb)] * ep[mono_q(tb)];
        }
        // (two spare entries: the second-half instantiation T0 = NT names monomials beyond
        // SFFT_MAX_T in code that only runs for TK = 10, NT = 5)
        double xsp[SFFT_MAX_DEG + 3] = {}, esp[SFFT_MAX_DEG + 3] = {};
        powers(xis, xsp);
        powers(etas, esp);
#pragma unroll
        for (int a = 0; a < NT; ++a) {
          const double wgt = rv[k] * xsp[mono_p(T0 + a)] * esp[mono_q(T0 + a)];
#pragma unroll
          for (int tb = 0; tb < TB; ++tb) acc[a][tb] = fma(wgt, q[tb], acc[a][tb]);
        }
      }
    }
  }
  if (active) {
#pragma unroll
    for (int a = 0; a < NT; ++a) {
      double* out = P.part + (((size_t)(blockIdx.x * P.nsub + sub) * P.TK + T0 + a) * P.L + s) * TB;
#pragma unroll
      for (int tb = 0; tb < TB; ++tb) out[tb] = acc[a][tb];
    }
  }
}

template <int NT, int TB>
__global__ void __launch_bounds__(KB_TH) k_kb_corr(KbParams P) {
  if (blockIdx.y == 0) kb_corr_body<NT, TB, 0>(P);
  else kb_corr_body<NT, TB, NT>(P);   // only TK = 10 is split in two halves of NT = 5
}

// kbCorr[(t*L + s)*TB + t'] = sum over the partials in a fixed order: 8 lanes per entry, each
// summing every 8th partial sequentially, then a shuffle tree.
__global__ void __launch_bounds__(256) k_kb_reduce(const double* __restrict__ part, double* corr, int npart, int n) {
  const int e = (blockIdx.x * 256 + threadIdx.x) >> 3, sl = threadIdx.x & 7;
  double a = 0.0;
  if (e < n)
    for (int k = sl; k < npart; k += 8) a += part[(size_t)k * n + e];
  a += __shfl_xor_sync(0xffffffffu, a, 1);
  a += __shfl_xor_sync(0xffffffffu, a, 2);
  a += __shfl_xor_sync(0xffffffffu, a, 4);
  if (e < n && sl == 0) corr[e] = a;
}

template <int NT, int TB>
static sfft_status launch_kb_corr_t(const KbParams& P, cudaStream_t st) {
  dim3 grid(SFFT_KB_NBLK, P.TK / NT, (P.L + KB_TH - 1) / KB_TH);
  k_kb_corr<NT, TB><<<grid, KB_TH, 0, st>>>(P);
  SFFT_LAUNCH_CHECK();
  return SFFT_OK;
}
template <int TB>
static sfft_status launch_kb_corr_tb(const KbParams& P, cudaStream_t st) {
  switch (P.TK) {
    case 1: return launch_kb_corr_t<1, TB>(P, st);
    case 3: return launch_kb_corr_t<3, TB>(P, st);
    case 6: return launch_kb_corr_t<6, TB>(P, st);
    case 10: return launch_kb_corr_t<5, TB>(P, st);
    default: return SFFT_ERR_UNSUPPORTED;
  }
}

sfft_status sfft_launch_kb(sfft_plan* p, const double* R, const unsigned char* mask, cudaStream_t st, int* nl) {
  const int H = p->H, W = p->W;
  const int rowsPerBlock = 8;
  k_sp_rows<false><<<(H + rowsPerBlock - 1) / rowsPerBlock, 32 * rowsPerBlock, 0, st>>>(mask, H, W, p->w, p->spCount, nullptr, nullptr, p->fmFlag);
  SFFT_LAUNCH_CHECK();
  k_sp_scan<<<1, 1024, 0, st>>>(p->spCount, p->spOff, H, p->fmFlag, p->fmList);
  SFFT_LAUNCH_CHECK();
  k_sp_rows<true><<<(H + rowsPerBlock - 1) / rowsPerBlock, 32 * rowsPerBlock, 0, st>>>(mask, H, W, p->w, p->spCount, p->spOff, p->spList, p->fmFlag);
  SFFT_LAUNCH_CHECK();
  KbParams P;
  P.R = R; P.mask = mask; P.spOff = p->spOff; P.spList = p->spList; P.part = p->kbPart;
  P.H = H; P.W = W; P.w = p->w; P.L = p->L; P.TK = p->TK; P.TB = p->TB;
  P.nsub = KB_TH / p->L;
  if (P.nsub < 1) P.nsub = 1;   // L > KB_TH: see kb_corr_body
  for (int t = 0; t < p->TK; ++t) { P.monoK[t][0] = p->monoK[t][0]; P.monoK[t][1] = p->monoK[t][1]; }
  for (int t = 0; t < p->TB; ++t) { P.monoB[t][0] = p->monoB[t][0]; P.monoB[t][1] = p->monoB[t][1]; }
  sfft_status rs;
  switch (p->TB) {
    case 1: rs = launch_kb_corr_tb<1>(P, st); break;
    case 3: rs = launch_kb_corr_tb<3>(P, st); break;
    case 6: rs = launch_kb_corr_tb<6>(P, st); break;
    case 10: rs = launch_kb_corr_tb<10>(P, st); break;
    default: rs = SFFT_ERR_UNSUPPORTED; break;
  }
  if (rs != SFFT_OK) return rs;
  const int n = p->TK * p->L * p->TB;
  k_kb_reduce<<<(8 * n + 255) / 256, 256, 0, st>>>(p->kbPart, p->kbCorr, SFFT_KB_NBLK * P.nsub, n);
  SFFT_LAUNCH_CHECK();
  *nl += 5;
  return SFFT_OK;
}
