// Exact unmasked-pixel objective, structured part: fully masked ROWS and COLUMNS.
//
// sfft_build_system_exact subtracts sum_{x masked} g(x) g(x)^T from the unmasked system.  A CCD's mask is
// mostly a frame of full border rows and columns; for a fully masked row y0 the sum over its pixels is
// a 1-D circular correlation along x,
//   sum_x R_t(x-u, y0-v) R_t'(x-u', y0-v') = eta(y0-v)^q eta(y0-v')^q' sum_x' [xi^p R](x', y0-v) [xi^p' R](x' + (u-u'), y0-v'),
// so all of it follows from the correlations  Q[A; B; d] = sum_n Z_A[n] Z_B[(n + d) mod Len],  |d| <= 2w,
// between a few "strips": the rows y0 - v of xi^p R (p <= DK), the rows y0 of S, and the polynomial rows
// xi^a (a <= DB) that give the kernel-background and background-background parts.  Fully masked columns
// are the transposed statement (strips along y, weights eta^q).  With a(y) = 1 on the full rows and
// b(x) = 1 on the full columns,
//   masked = a + b - a b + rest:   rows term + columns term - corners (pixel list, added back) + rest (pixel list),
// and only `rest` and the corners go through the dense rank-K update of k_exact.cu -- nothing at all for
// a pure frame mask (73 584 pixels at the full CCD).
//
// Everything is sized on the device (the calls never synchronise): at most XS_MAXT fully masked target
// lines and XS_MAXS distinct source lines per direction take this path, further full lines simply stay
// in the pixel list.  All sums have a fixed order.
//   k_xs_colcount   masked pixels per column (integer atomics)
//   k_xs_plan       accepted full rows / columns, their source lines, flags for the list kernels
//   k_xs_list       ordered pixel lists: `rest` (masked, outside the accepted lines) and corners
//   k_xs_gather     the strips Z (R lines x powers, S lines, polynomial lines)
//   k_xs_corr       Q[A][B][d]
//   k_xs_scatter    A, b -= the lines' terms (both triangles from one sum: A stays bitwise symmetric)
#include "sfft_common.cuh"

#define XS_MAXT SFFT_XS_MAXT
#define XS_MAXS SFFT_XS_MAXS
#define XS_NP (SFFT_MAX_DEG + 1)          // powers per line
#define XS_NR (XS_MAXS * XS_NP)           // R strips
#define XS_NSTRIP (XS_NR + XS_MAXT + XS_NP)   // + S strips + polynomial strips
#define XS_NA (XS_NR + XS_NP)             // A side of the correlations: R strips and polynomial strips
#define XS_LAGS (2 * 2 * SFFT_XS_MAXW + 1)

// per-direction plan, device resident
struct XsPlan {
  int nT, nS;
  int tgt[XS_MAXT];     // accepted fully masked lines
  int src[XS_MAXS];     // distinct source lines (tgt - shift, wrapped)
};

size_t sfft_xs_plan_bytes() { return 2 * sizeof(XsPlan); }
size_t sfft_xs_strip_bytes(int H, int W) { return (size_t)XS_NSTRIP * (size_t)(H > W ? H : W) * sizeof(double); }
size_t sfft_xs_q_bytes() { return (size_t)XS_NA * XS_NSTRIP * XS_LAGS * sizeof(double); }

__global__ void __launch_bounds__(256) k_xs_colcount(const unsigned char* __restrict__ mask, int H, int W, int* colcnt) {
  const int x = blockIdx.x * 256 + threadIdx.x;
  if (x >= W) return;
  const int y0 = blockIdx.y * 64, y1 = min(H, y0 + 64);
  int c = 0;
  for (int y = y0; y < y1; ++y) c += mask[(size_t)y * W + x] ? 1 : 0;
  if (c) atomicAdd(colcnt + x, c);
}

// One CTA.  dir 0: rows (cnt = rowcnt, M = H lines, full when cnt == W); dir 1: columns.
// flag[line] = 1 for accepted full lines; srcIdx[line] = index into src or -1.  The full lines are found
// in parallel (ordered compaction by a block scan), the few candidates are then accepted one after the
// other by one thread per direction on shared-memory copies of the index arrays.
#define XS_MAXC 128   // full lines looked at per direction
__global__ void __launch_bounds__(1024) k_xs_plan(const int* __restrict__ rowcnt, const int* __restrict__ colcnt, int H, int W,
                                                  int w, int maxT, XsPlan* plans, unsigned char* rowFull, unsigned char* colFull,
                                                  int* srcIdxY, int* srcIdxX) {
  extern __shared__ int xs_sm[];
  int* sY = xs_sm;              // [H]
  int* sX = xs_sm + H;          // [W]
  __shared__ int part[1024];
  __shared__ int cand[2][XS_MAXC];
  __shared__ int ncand[2];
  __shared__ XsPlan sp[2];
  const int tid = threadIdx.x;
  for (int i = tid; i < H; i += 1024) sY[i] = -1;
  for (int i = tid; i < W; i += 1024) sX[i] = -1;
  for (int dir = 0; dir < 2; ++dir) {
    const int M = dir ? W : H, fullv = dir ? H : W;
    const int* cnt = dir ? colcnt : rowcnt;
    const int per = (M + 1023) / 1024;
    int mine = 0;
    for (int i = 0; i < per; ++i) {
      const int l = tid * per + i;
      if (l < M && cnt[l] == fullv) ++mine;
    }
    part[tid] = mine;
    __syncthreads();
    for (int o = 1; o < 1024; o <<= 1) {
      const int t = tid >= o ? part[tid - o] : 0;
      __syncthreads();
      part[tid] += t;
      __syncthreads();
    }
    int pos = part[tid] - mine;
    for (int i = 0; i < per; ++i) {
      const int l = tid * per + i;
      if (l < M && cnt[l] == fullv) { if (pos < XS_MAXC) cand[dir][pos] = l; ++pos; }
    }
    if (tid == 1023) ncand[dir] = part[1023] < XS_MAXC ? part[1023] : XS_MAXC;
    __syncthreads();
  }
  if (tid == 0 || tid == 32) {
    const int dir = tid ? 1 : 0;
    const int M = dir ? W : H;
    int* sidx = dir ? sX : sY;
    XsPlan& P = sp[dir];
    int nT = 0, nS = 0;
    for (int ic = 0; ic < ncand[dir] && nT < maxT; ++ic) {
      const int l = cand[dir][ic];
      int need = 0;
      for (int s = -w; s <= w; ++s) need += sidx[(l - s + M) % M] < 0 ? 1 : 0;
      if (nS + need > XS_MAXS) continue;
      for (int s = -w; s <= w; ++s) {
        const int ls = (l - s + M) % M;
        if (sidx[ls] < 0) { sidx[ls] = nS; P.src[nS++] = ls; }
      }
      P.tgt[nT++] = l;
    }
    P.nT = nT; P.nS = nS;
  }
  __syncthreads();
  for (int i = tid; i < H; i += 1024) { srcIdxY[i] = sY[i]; rowFull[i] = 0; }
  for (int i = tid; i < W; i += 1024) { srcIdxX[i] = sX[i]; colFull[i] = 0; }
  __syncthreads();
  for (int dir = 0; dir < 2; ++dir) {
    for (int k = tid; k < sp[dir].nT; k += 1024) (dir ? colFull : rowFull)[sp[dir].tgt[k]] = 1;
    for (int i = tid; i < (int)(sizeof(XsPlan) / sizeof(int)); i += 1024)
      reinterpret_cast<int*>(plans + dir)[i] = reinterpret_cast<const int*>(&sp[dir])[i];
  }
}

// Ordered pixel lists, one warp per row, 16 pixels per lane and step (W is a multiple of 32).
// MODE 1: masked pixels outside the accepted full rows and columns; MODE 2: corners (accepted row AND column).
template <bool FILL, int MODE>
__global__ void __launch_bounds__(256) k_xs_list(const unsigned char* __restrict__ mask, const unsigned char* __restrict__ rowFull,
                                                 const unsigned char* __restrict__ colFull, int H, int W, int* cnt,
                                                 const int* __restrict__ off, int* list) {
  const int lane = threadIdx.x & 31;
  const int y = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (y >= H) return;
  const bool rf = rowFull[y] != 0;
  const int base = FILL ? off[y] : 0;
  int total = 0;
  for (int k = 0; k < (W + 511) / 512; ++k) {   // uniform trip count for the shuffles
    const int x0 = k * 512 + lane * 16;
    unsigned mk = 0u;
    if (x0 < W && (MODE == 1 ? !rf : rf)) {
      const uint4 m16 = *reinterpret_cast<const uint4*>(mask + (size_t)y * W + x0);
      const uint4 c16 = *reinterpret_cast<const uint4*>(colFull + x0);
      const unsigned wm[4] = {m16.x, m16.y, m16.z, m16.w}, wc[4] = {c16.x, c16.y, c16.z, c16.w};
#pragma unroll
      for (int q = 0; q < 4; ++q)
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          const bool m = ((wm[q] >> (8 * i)) & 0xffu) != 0u, cf = ((wc[q] >> (8 * i)) & 0xffu) != 0u;
          if (MODE == 1 ? (m && !cf) : cf) mk |= 1u << (4 * q + i);
        }
    }
    const int c = __popc(mk);
    int incl = c;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int t = __shfl_up_sync(0xffffffffu, incl, o);
      if (lane >= o) incl += t;
    }
    if (FILL) {
      int pos = base + total + incl - c;
      while (mk) {
        const int i = __ffs(mk) - 1;
        mk &= mk - 1;
        list[pos++] = y * W + x0 + i;
      }
    }
    total += __shfl_sync(0xffffffffu, incl, 31);
  }
  if (!FILL && lane == 0) cnt[y] = total;
}

struct XsParams {
  const double* R;
  const double* S;
  const XsPlan* plan;       // the direction's plan
  const int* srcIdx;        // line -> source index
  double* Z;                // [XS_NSTRIP][Len]
  double* Q;                // [XS_NA][XS_NSTRIP][XS_LAGS]
  double* A;
  double* b;
  int H, W, w, L, TK, TB, N, DK, DB;
  int cols;                 // 0: rows (strips along x), 1: columns (strips along y)
  int monoK[SFFT_MAX_T][2], monoB[SFFT_MAX_T][2];
};

// strip index helpers
__device__ __forceinline__ int xs_r(int line, int pw) { return line * XS_NP + pw; }
__device__ __forceinline__ int xs_s(int k) { return XS_NR + k; }
__device__ __forceinline__ int xs_p(int a) { return XS_NR + XS_MAXT + a; }
// A-side index (R strips, then polynomial strips)
__device__ __forceinline__ int xs_a_of_strip(int strip) { return strip < XS_NR ? strip : XS_NR + (strip - XS_NR - XS_MAXT); }

// blockIdx.y = strip; builds Z[strip][n]
__global__ void __launch_bounds__(256) k_xs_gather(XsParams P) {
  const int Len = P.cols ? P.H : P.W;
  const int n = blockIdx.x * 256 + threadIdx.x;
  const int strip = blockIdx.y;
  if (n >= Len) return;
  const XsPlan& pl = *P.plan;
  const double c = (double)(2 * n + 1 - Len) / (double)Len;     // along coordinate (xi for rows, eta for columns)
  double v;
  if (strip < XS_NR) {
    const int line = strip / XS_NP, pw = strip - line * XS_NP;
    if (line >= pl.nS || pw > P.DK) return;
    const int l = pl.src[line];
    const double r = P.cols ? P.R[(size_t)n * P.W + l] : P.R[(size_t)l * P.W + n];
    v = r * ipow(c, pw);
  } else if (strip < XS_NR + XS_MAXT) {
    const int k = strip - XS_NR;
    if (k >= pl.nT) return;
    const int l = pl.tgt[k];
    v = P.cols ? P.S[(size_t)n * P.W + l] : P.S[(size_t)l * P.W + n];
  } else {
    const int a = strip - XS_NR - XS_MAXT;
    if (a > P.DB) return;
    v = ipow(c, a);
  }
  P.Z[(size_t)strip * Len + n] = v;
}

// active strip?
__device__ __forceinline__ bool xs_active(const XsParams& P, const XsPlan& pl, int strip) {
  if (strip < XS_NR) { const int line = strip / XS_NP, pw = strip - line * XS_NP; return line < pl.nS && pw <= P.DK; }
  if (strip < XS_NR + XS_MAXT) return strip - XS_NR < pl.nT;
  return strip - XS_NR - XS_MAXT <= P.DB;
}

// Q[a][B][d] = sum_n Z_A[n] Z_B[(n + d) mod Len], d = -2w .. 2w at index d + 2w.  blockIdx.x = B strip: the whole
// CTA slides its window over the SAME Z_B (it stays in L1), every WARP takes its own A strips (A-side index
// blockIdx.y * 8 + warp, then strided) and reads each Z_A element once; a lane takes runs of 4 consecutive n
// (a warp reads 1 KB contiguous per step, 128-bit loads).  The 2 * 2w + 1 sums are reduced by a shuffle tree
// (fixed order), no block barrier.  R x R pairs: Q[A;B;d] = Q[B;A;-d], only A <= B is computed.
#define XS_CORR_ACH 4   // A chunks (gridDim.y)
__global__ void __launch_bounds__(256) k_xs_corr(XsParams P) {
  constexpr int NL = XS_LAGS, DM = 2 * SFFT_XS_MAXW;
  const int Len = P.cols ? P.H : P.W;
  const XsPlan& pl = *P.plan;
  const int sb = blockIdx.x;
  if (!xs_active(P, pl, sb)) return;
  const int D = 2 * P.w;
  const int lane = threadIdx.x & 31, wrp = threadIdx.x >> 5;
  const double* ZB = P.Z + (size_t)sb * Len;
  for (int ia = blockIdx.y * 8 + wrp; ia < XS_NA; ia += 8 * gridDim.y) {
    const int sa = ia < XS_NR ? ia : XS_NR + XS_MAXT + (ia - XS_NR);
    if (!xs_active(P, pl, sa)) continue;
    if (sb < XS_NR && sa < XS_NR && sb < sa) continue;
    const double* ZA = P.Z + (size_t)sa * Len;
    double acc[NL];
#pragma unroll
    for (int d = 0; d < NL; ++d) acc[d] = 0.0;
    // the window of Z_B starts at n0 - DM (even, so pairs never straddle the wrap)
    for (int n0 = lane * 4; n0 < Len; n0 += 32 * 4) {
      double a[4], bw[4 + 2 * DM];
#pragma unroll
      for (int i = 0; i < 4; i += 2) {
        const double2 t = *reinterpret_cast<const double2*>(ZA + n0 + i);
        a[i] = t.x; a[i + 1] = t.y;
      }
#pragma unroll
      for (int i = 0; i < 4 + 2 * DM; i += 2) {
        int m = n0 - DM + i;
        m = m < 0 ? m + Len : (m >= Len ? m - Len : m);      // Len >= 32 > DM: one wrap at most
        const double2 t = *reinterpret_cast<const double2*>(ZB + m);
        bw[i] = t.x; bw[i + 1] = t.y;
      }
#pragma unroll
      for (int d = 0; d < NL; ++d)
#pragma unroll
        for (int i = 0; i < 4; ++i) acc[d] = fma(a[i], bw[i + d], acc[d]);
    }
#pragma unroll
    for (int d = 0; d < NL; ++d) {
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) acc[d] += __shfl_xor_sync(0xffffffffu, acc[d], o);
    }
    // acc index d <-> lag (d - DM); stored at lag + D of the plan's own range when |lag| <= D
#pragma unroll
    for (int d = 0; d < NL; ++d) {
      const int lag = d - DM;
      if (lane == (d & 31) && lag >= -D && lag <= D) P.Q[((size_t)ia * XS_NSTRIP + sb) * NL + lag + D] = acc[d];
    }
  }
}

// A, b -= the accepted lines' terms.  One thread per entry (i >= j) of the system with b as row N.
__global__ void __launch_bounds__(256) k_xs_scatter(XsParams P) {
  const int N = P.N, nK = P.L * P.TK, S1 = 2 * P.w + 1, D = 2 * P.w;
  const size_t total = (size_t)(N + 1) * (N + 2) / 2 - 1;   // lower triangle of the (N+1) x (N+1) system without its corner
  const size_t e = (size_t)blockIdx.x * 256 + threadIdx.x;
  if (e >= total) return;
  const XsPlan& pl = *P.plan;
  if (pl.nT == 0) return;
  int i = (int)((sqrt(8.0 * (double)e + 1.0) - 1.0) * 0.5);
  while ((size_t)(i + 1) * (i + 2) / 2 <= e) ++i;
  while ((size_t)i * (i + 1) / 2 > e) --i;
  const int j = (int)(e - (size_t)i * (i + 1) / 2);
  const int M = P.cols ? P.W : P.H;                          // lines of this direction
  const double invM = 1.0 / (double)M;
  // column kinds: 1 kernel (along shift a, cross shift c, along power ap, cross power cp), 2 background, 3 S
  auto decode = [&](int n, int& kind, int& a, int& c, int& ap, int& cp) {
    if (n < nK) {
      const int t = n / P.L, s = n - t * P.L;
      const int u = s % S1 - P.w, v = s / S1 - P.w, p = P.monoK[t][0], q = P.monoK[t][1];
      kind = 1;
      if (P.cols) { a = v; c = u; ap = q; cp = p; } else { a = u; c = v; ap = p; cp = q; }
    } else if (n < N) {
      const int p = P.monoB[n - nK][0], q = P.monoB[n - nK][1];
      kind = 2; a = c = 0;
      if (P.cols) { ap = q; cp = p; } else { ap = p; cp = q; }
    } else {
      kind = 3; a = c = ap = cp = 0;
    }
  };
  int ki, ai, ci, api, cpi, kj, aj, cj, apj, cpj;
  decode(i, ki, ai, ci, api, cpi);
  decode(j, kj, aj, cj, apj, cpj);
  // j <= i and the kinds are ordered (kernel < background < S), so kj <= ki
  const double* Q = P.Q;
  auto q_at = [&](int sA, int sB, int lag) -> double {
    if (sA < XS_NR && sB < XS_NR && sB < sA) { const int t = sA; sA = sB; sB = t; lag = -lag; }   // R x R: stored for A <= B
    return Q[((size_t)xs_a_of_strip(sA) * XS_NSTRIP + sB) * XS_LAGS + lag + D];
  };
  double sum = 0.0;
  for (int k = 0; k < pl.nT; ++k) {
    const int tk = pl.tgt[k];
    const double ct = (double)(2 * tk + 1 - M) * invM;      // cross coordinate of the target line
    double term;
    if (kj == 1) {
      const int lj = (tk - cj + M) % M;
      const double wj = ipow((double)(2 * lj + 1 - M) * invM, cpj);
      const int sj = xs_r(P.srcIdx[lj], apj);
      if (ki == 1) {          // kernel-kernel: Q[R_i; R_j; d = a_i - a_j]
        const int li = (tk - ci + M) % M;
        const double wi = ipow((double)(2 * li + 1 - M) * invM, cpi);
        term = wi * wj * q_at(xs_r(P.srcIdx[li], api), sj, ai - aj);
      } else if (ki == 2) {   // background(i) x kernel(j): sum_n' Z_Rj[n'] P_i[n' + a_j]
        term = ipow(ct, cpi) * wj * q_at(sj, xs_p(api), aj);
      } else {                // S x kernel(j): sum_n' Z_Rj[n'] S[n' + a_j]
        term = wj * q_at(sj, xs_s(k), aj);
      }
    } else if (kj == 2) {
      if (ki == 2) term = ipow(ct, cpi + cpj) * q_at(xs_p(api), xs_p(apj), 0);
      else term = ipow(ct, cpj) * q_at(xs_p(apj), xs_s(k), 0);   // S x background(j)
    } else {
      term = 0.0;   // (S, S) is not part of the system
    }
    sum += term;
  }
  if (ki == 3) {
    P.b[j] -= sum;
  } else {
    P.A[(size_t)i * N + j] -= sum;
    if (i != j) P.A[(size_t)j * N + i] -= sum;
  }
}

// ---- host side ---------------------------------------------------------------------------------------
sfft_status sfft_launch_exact_syrk(sfft_plan* p, const double* R, const double* S, const int* list, const int* off,
                                   double* A, double* b, double sign, cudaStream_t st, int* nl);
void sfft_launch_mk_scan(const int* cnt, int* off, int H, cudaStream_t st);

sfft_status sfft_launch_exact_update(sfft_plan* p, const double* R, const double* S, const unsigned char* mask,
                                     double* A, double* b, cudaStream_t st, int* nl) {
  const int H = p->H, W = p->W, rowsPerBlock = 8;
  const int rowBlocks = (H + rowsPerBlock - 1) / rowsPerBlock;
  XsPlan* plans = reinterpret_cast<XsPlan*>(p->xsPlan);
  // 1. masked pixels per row and per column, the accepted full lines (none for w > SFFT_XS_MAXW, whose lag
  //    range the strip correlations are not compiled for: every masked pixel then takes the rank-K update)
  SFFT_CUDA_TRY(cudaMemsetAsync(p->xsColCnt, 0, sizeof(int) * (size_t)W, st));
  k_xs_colcount<<<dim3((W + 255) / 256, (H + 63) / 64), 256, 0, st>>>(mask, H, W, p->xsColCnt);
  SFFT_LAUNCH_CHECK();
  // (row counts: the all-masked-pixels count of MODE 1 with no line accepted yet == plain masked count)
  SFFT_CUDA_TRY(cudaMemsetAsync(p->xsRowFull, 0, (size_t)H, st));
  SFFT_CUDA_TRY(cudaMemsetAsync(p->xsColFull, 0, (size_t)W, st));
  k_xs_list<false, 1><<<rowBlocks, 32 * rowsPerBlock, 0, st>>>(mask, p->xsRowFull, p->xsColFull, H, W, p->spCount, nullptr, nullptr);
  SFFT_LAUNCH_CHECK();
  k_xs_plan<<<1, 1024, sizeof(int) * (size_t)(H + W), st>>>(p->spCount, p->xsColCnt, H, W, p->w, p->w <= SFFT_XS_MAXW ? XS_MAXT : 0, plans, p->xsRowFull, p->xsColFull, p->xsSrcIdxY, p->xsSrcIdxX);
  SFFT_LAUNCH_CHECK();
  *nl += 3;
  // 2. the two directions' strips, correlations and terms
  for (int dir = 0; dir < 2; ++dir) {
    XsParams P;
    P.R = R; P.S = S; P.plan = plans + dir; P.srcIdx = dir ? p->xsSrcIdxX : p->xsSrcIdxY;
    P.Z = p->xsZ; P.Q = p->xsQ; P.A = A; P.b = b;
    P.H = H; P.W = W; P.w = p->w; P.L = p->L; P.TK = p->TK; P.TB = p->TB; P.N = p->N; P.DK = p->DK; P.DB = p->DB;
    P.cols = dir;
    for (int t = 0; t < p->TK; ++t) { P.monoK[t][0] = p->monoK[t][0]; P.monoK[t][1] = p->monoK[t][1]; }
    for (int t = 0; t < p->TB; ++t) { P.monoB[t][0] = p->monoB[t][0]; P.monoB[t][1] = p->monoB[t][1]; }
    const int Len = dir ? H : W;
    k_xs_gather<<<dim3((Len + 255) / 256, XS_NSTRIP), 256, 0, st>>>(P);
    SFFT_LAUNCH_CHECK();
    k_xs_corr<<<dim3(XS_NSTRIP, XS_CORR_ACH), 256, 0, st>>>(P);
    SFFT_LAUNCH_CHECK();
    const size_t total = (size_t)(p->N + 1) * (p->N + 2) / 2 - 1;
    k_xs_scatter<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(P);
    SFFT_LAUNCH_CHECK();
    *nl += 3;
  }
  // 3. pixel lists: the masked pixels outside the accepted lines (subtracted), the corners (added back)
  k_xs_list<false, 1><<<rowBlocks, 32 * rowsPerBlock, 0, st>>>(mask, p->xsRowFull, p->xsColFull, H, W, p->spCount, nullptr, nullptr);
  SFFT_LAUNCH_CHECK();
  sfft_launch_mk_scan(p->spCount, p->spOff, H, st);
  SFFT_LAUNCH_CHECK();
  k_xs_list<true, 1><<<rowBlocks, 32 * rowsPerBlock, 0, st>>>(mask, p->xsRowFull, p->xsColFull, H, W, p->spCount, p->spOff, p->spList);
  SFFT_LAUNCH_CHECK();
  *nl += 3;
  sfft_status s = sfft_launch_exact_syrk(p, R, S, p->spList, p->spOff, A, b, -1.0, st, nl);
  if (s != SFFT_OK) return s;
  k_xs_list<false, 2><<<rowBlocks, 32 * rowsPerBlock, 0, st>>>(mask, p->xsRowFull, p->xsColFull, H, W, p->xsCnt, nullptr, nullptr);
  SFFT_LAUNCH_CHECK();
  sfft_launch_mk_scan(p->xsCnt, p->xsOff, H, st);
  SFFT_LAUNCH_CHECK();
  k_xs_list<true, 2><<<rowBlocks, 32 * rowsPerBlock, 0, st>>>(mask, p->xsRowFull, p->xsColFull, H, W, p->xsCnt, p->xsOff, p->xsList);
  SFFT_LAUNCH_CHECK();
  *nl += 3;
  return sfft_launch_exact_syrk(p, R, S, p->xsList, p->xsOff, A, b, +1.0, st, nl);
}
