// Column direction of the system build without any full-length column transform (north_star
// subsystems (2),(3)): the cross-correlation maps are needed only at the lags
// |dy| <= D (D = 2w <= 10), so the sum over y is cut into blocks and every block is correlated with a
// SHORT transform,
//
//   sum_y conj(f[y]) g[y+dy]  =  sum_blocks  sum_{y in block} conj(f[y]) g[y+dy],      |dy| <= D.
//
// With CB_N = 128 and B = CB_N - 2D, block i owns the "centre" rows [iB, iB+B) and reads the "extended"
// rows [iB-D, iB+B+D) (mod H).  c = f restricted to the centre rows and e = g on the extended rows, both
// placed on the same 128-point grid, have the block's correlation as their 128-point CIRCULAR
// correlation at |dy| <= D (no wrap: the centre rows sit D points inside the grid), i.e. in the
// frequency domain  conj(C_f[k]) E_g[k].  These products are simply ADDED over the blocks of a column,
// and one 128-point inverse per pair and column, evaluated only at the 2D+1 lags, ends the column:
//
//   Y[dy][kx] = H sum_y conj(f) g(y+dy) = (H/128) sum_k e^{+2 pi i k dy/128} sum_blocks conj(C_f[k]) E_g[k].
//
// Against the full-length formulation (one 2048-point FFT per spectrum, products, pruned inverse with
// 2D+1 twiddled accumulations per 8 frequencies) this needs 1.6x fewer fp64 operations at the full
// CCD, and a third of them become plain complex multiply-accumulates.  The sequences are the column kx
// of the row spectra T (k_row_fwd), f = eta^q T_p for every kernel monomial t = (p,q) ("centre" AND
// "extended" version: 2 TK sequences) and g = the row spectrum of m S ("extended" only).
//
// One CTA per SM (persistent, columns round-robin), 384 threads (three warps per scheduler, so a thread
// may hold 168 registers), a stage = up to CB_G = 7 blocks whose 2TK+1 sequences sit in shared memory
// (182 KB at DK = 2).  With one column in flight per SM the column's 27 x 128 complex accumulators cost
// 36 registers per thread (a third of the pairs each), which leaves room for the radix-16 butterflies:
//   phase 1  warp = (group g < 3, pair of blocks), half warp = one block, lane j < 16.  A group owns a
//            compile-time list of the block's sequences (5, 5 and 3 of the 13 at DK = 2) that reads at most
//            two row images; their 8 x 16 block elements (n = j + 16 r) were requested during phase 3 of
//            the stage before (the first image into registers, the second by cp.async into a staging slot).  Per sequence: eta^q weighting, zero padding, radix-8 butterfly over r,
//            twiddle w128^(j k1), store.  Both halves of a warp run the same list: no divergence;
//   phase 2  radix-16 butterflies over j for every (block, sequence, k1): X[k1 + 8 k2];
//   phase 3  thread = (frequency k, third of the pairs): the stage's products accumulate in registers
//            (6-7 operand loads per 9 pairs);
//   phase 4  (once per column) accumulators -> shared memory, 16-point inverse over b (k = a + 8 b),
//            then the 2D+1 lags of every pair (8 twiddled terms each), Y[pair][dy][kx].
// Shared-memory positions are XOR-swizzled (slot k1*16 + (j ^ k1)): every pass is conflict free with no
// padding.  T has the row-group layout T[img][y/G][kx][y%G], G = SFFT_T_G = 8 (k_row2_fwd): a half warp's 16
// rows of a column are two whole 128-byte lines.
#include <math.h>
#include "fft_smem.cuh"

#define CB_N 128          // block transform length
#define CB_TH 384         // 12 warps = 3 per scheduler: 168 registers per thread
#define CB_G 7            // most blocks per stage (shared memory)
#define CB_LAGS 21        // 2 * 10 + 1

struct ColbParams {
  const cplx* T;          // [nimg][H/G][NC+1][G] row spectra, row-group layout (G = SFFT_T_G)
  cplx* Y;                // [nPair][nLag][pitch]
  const PairDesc* pairs;
  const cplx* tw128;      // e^{-2 pi i m/128}, m < 128
  int H, NC, pitch, nLag, nPair, nimg;
  int D;                  // lag half-range (halo)
  int B;                  // centre rows per block = CB_N - 2 D
  int nblk;               // blocks per column = ceil(H / B)
  int nst;                // stages per column = ceil(nblk / CB_G); stage i holds blocks [i nblk/nst, (i+1) nblk/nst)
};

// Phase-1 job lists.  Sequence index: centre version of monomial t at t, extended version at TK + t,
// S~ (extended only) at 2 TK.  Monomial order (p,q): DK = 2: (0,0),(1,0),(0,1),(2,0),(1,1),(0,2); DK = 1:
// (0,0),(1,0),(0,1); row image = p, q = power of eta.  A job = (buffer 0/1, q, centre?, sequence); group
// g reads row image IMG[g][0] into buffer 0 and IMG[g][1] into buffer 1 (-1: none); the extended
// sequences of an image come before its centre ones.
template <int TK> struct CbP1;
template <> struct CbP1<6> {
  static constexpr int N[3] = {5, 5, 3};
  static constexpr int IMG[3][2] = {{0, -1}, {1, 3}, {0, 2}};
  //                                   E(0,0)      E(0,1)      E(0,2)       C(0,0)     C(0,1)
  static constexpr int BUF[3][5] = {{0, 0, 0, 0, 0}, {0, 0, 0, 0, 1}, {0, 1, 1, 0, 0}};
  static constexpr int Q[3][5] = {{0, 1, 2, 0, 1}, {0, 1, 0, 1, 0}, {2, 0, 0, 0, 0}};
  static constexpr int CEN[3][5] = {{0, 0, 0, 1, 1}, {0, 0, 1, 1, 0}, {1, 0, 1, 0, 0}};
  static constexpr int SEQ[3][5] = {{6, 8, 11, 0, 2}, {7, 10, 1, 4, 12}, {5, 9, 3, 0, 0}};
};
template <> struct CbP1<3> {
  static constexpr int N[3] = {4, 3, 0};
  static constexpr int IMG[3][2] = {{0, -1}, {1, 2}, {-1, -1}};
  static constexpr int BUF[3][5] = {{0, 0, 0, 0, 0}, {0, 0, 1, 0, 0}, {0, 0, 0, 0, 0}};
  static constexpr int Q[3][5] = {{0, 1, 0, 1, 0}, {0, 0, 0, 0, 0}, {0, 0, 0, 0, 0}};
  static constexpr int CEN[3][5] = {{0, 0, 1, 1, 0}, {0, 1, 0, 0, 0}, {0, 0, 0, 0, 0}};
  static constexpr int SEQ[3][5] = {{3, 5, 0, 2, 0}, {4, 1, 6, 0, 0}, {0, 0, 0, 0, 0}};
};
template <> struct CbP1<1> {
  static constexpr int N[3] = {2, 1, 0};
  static constexpr int IMG[3][2] = {{0, -1}, {1, -1}, {-1, -1}};
  static constexpr int BUF[3][5] = {{0, 0, 0, 0, 0}, {0, 0, 0, 0, 0}, {0, 0, 0, 0, 0}};
  static constexpr int Q[3][5] = {{0, 0, 0, 0, 0}, {0, 0, 0, 0, 0}, {0, 0, 0, 0, 0}};
  static constexpr int CEN[3][5] = {{0, 1, 0, 0, 0}, {0, 0, 0, 0, 0}, {0, 0, 0, 0, 0}};
  static constexpr int SEQ[3][5] = {{1, 0, 0, 0, 0}, {2, 0, 0, 0, 0}, {0, 0, 0, 0, 0}};
};

// Pair partition for phase 3.  Part (T0, T1, U0, U1) owns the pairs (t, t2), T0 <= t < T1,
// max(t, U0) <= t2 <= U1 (t2 = TK stands for S~).  For TK = 6 the three parts hold 9 pairs each and
// read 7, 6 and 7 operands: (C0-2 x E0-3), (C0-2 x E4,5,S), (C3-5 x E3,4,5,S).
template <int TK> struct CbParts;
template <> struct CbParts<6> { static constexpr int T0[3] = {0, 0, 3}, T1[3] = {3, 3, 6}, U0[3] = {0, 4, 3}, U1[3] = {3, 6, 6}; };
template <> struct CbParts<3> { static constexpr int T0[3] = {0, 1, 2}, T1[3] = {1, 2, 3}, U0[3] = {0, 1, 2}, U1[3] = {3, 3, 3}; };
template <> struct CbParts<1> { static constexpr int T0[3] = {0, 0, 0}, T1[3] = {1, 0, 0}, U0[3] = {0, 0, 0}, U1[3] = {1, 0, 0}; };
__host__ __device__ constexpr int cb_max(int a, int b) { return a > b ? a : b; }
__host__ __device__ constexpr int cb_part_pairs(int T0, int T1, int U0, int U1) {
  int n = 0;
  for (int t = T0; t < T1; ++t)
    for (int t2 = cb_max(t, U0); t2 <= U1; ++t2) ++n;
  return n;
}

// offset of row y inside one image of T (column 0): T[img][y/G][kx][y%G], G = SFFT_T_G
__device__ __forceinline__ size_t cb_toff(int y, size_t grpStride) {
  return (size_t)(y / SFFT_T_G) * grpStride + (size_t)(y % SFFT_T_G);
}
__device__ __forceinline__ int cb_slot(int k1, int j) { return k1 * 16 + (j ^ k1); }   // k1 < 8, j < 16

// Phase 3 for one block: acc[] += conj(C_t) E_t2 over the part's pairs, every operand read once.
template <int TK, int T0, int T1, int U0, int U1>
__device__ __forceinline__ void cb_accumulate(cplx* acc, const cplx* __restrict__ ub, int pk) {
  cplx C[TK], E[TK + 1];
#pragma unroll
  for (int t = T0; t < T1; ++t) C[t] = ub[t * CB_N + pk];
#pragma unroll
  for (int t2 = cb_max(T0, U0); t2 <= U1; ++t2) E[t2] = ub[(TK + t2) * CB_N + pk];
  int idx = 0;
#pragma unroll
  for (int t = T0; t < T1; ++t) {
#pragma unroll
    for (int t2 = cb_max(t, U0); t2 <= U1; ++t2) {
      cfmac(acc[idx], C[t], E[t2]);
      ++idx;
    }
  }
}

// Phase 4a: the part's accumulators -> shared memory acs[pair][k] (pair index of the plan's list:
// kernel-kernel pairs (t <= t2) row-major upper-triangular, then (t, S) at nKK + t)
template <int TK, int T0, int T1, int U0, int U1>
__device__ __forceinline__ void cb_flush(const cplx* acc, cplx* acs, int k) {
  constexpr int NKK = TK * (TK + 1) / 2;
  int idx = 0;
#pragma unroll
  for (int t = T0; t < T1; ++t) {
#pragma unroll
    for (int t2 = cb_max(t, U0); t2 <= U1; ++t2) {
      const int pair = (t2 < TK) ? (t * TK - t * (t - 1) / 2 + (t2 - t)) : (NKK + t);
      acs[pair * CB_N + k] = acc[idx];
      ++idx;
    }
  }
}

// eta of the rows n = j + 16 r of a block: eta_r = e0 + r (32/H) for the unwrapped row, and -/+ 2 where the
// row index wrapped around the frame (only the halo of a column's first and last block does); every
// value is a multiple of 1/H, so the arithmetic is exact.
struct CbRows {
  double e0, step;
  unsigned cenbits;   // bit r: element r lies in the block's centre rows
  unsigned lobits;    // bit r: row index below 0 before wrapping (eta + 2)
  unsigned hibits;    // bit r: row index >= H before wrapping (eta - 2)
};
__device__ __forceinline__ double cb_eta(const CbRows& R, int r) {
  double e = fma((double)r, R.step, R.e0);
  if ((R.lobits >> r) & 1u) e += 2.0;
  if ((R.hibits >> r) & 1u) e -= 2.0;
  return e;
}

// One phase-1 job: sequence = DFT8 over r of (x[r] * eta_r^Q, zero outside the centre rows when CEN),
// twiddled by w128^(j k1) (table row k1 - 1 of s_w, lane j) and stored at the lane's slots of `dst`.
template <int Q, bool CEN>
__device__ __forceinline__ void cb_job(const cplx* x, const CbRows& R, cplx* dst, int j, const cplx* __restrict__ swj) {
  cplx v[8];
#pragma unroll
  for (int r = 0; r < 8; ++r) {
    if (Q == 0) {
      v[r] = x[r];
    } else {
      const double e = cb_eta(R, r);
      v[r] = cscale(x[r], Q == 1 ? e : e * e);
    }
    if (CEN && !((R.cenbits >> r) & 1u)) v[r] = cmake(0.0, 0.0);
  }
  Dft<8, -1>::run(v);
  dst[cb_slot(0, j)] = v[0];
#pragma unroll
  for (int k1 = 1; k1 < 8; ++k1) dst[cb_slot(k1, j)] = cmul(v[k1], swj[(k1 - 1) * 16]);
}

// the whole job list of group G on one block (ub = the block's sequences in shared memory).  x holds the
// group's first row image; its second one was staged in shared memory (xs, the lane's own 8 elements
// 16 apart) and replaces x when the list reaches its first buffer-1 job.
template <int TK, int G, int E>
__device__ __forceinline__ void cb_group_jobs(cplx* x, const cplx* xs, const CbRows& R, cplx* ub, int j,
                                              const cplx* __restrict__ swj) {
  using T = CbP1<TK>;
  if constexpr (E < T::N[G]) {
    if constexpr (T::BUF[G][E] == 1 && (E == 0 || T::BUF[G][E > 0 ? E - 1 : 0] == 0)) {
#pragma unroll
      for (int r = 0; r < 8; ++r) x[r] = xs[16 * r];
    }
    cb_job<T::Q[G][E], T::CEN[G][E] != 0>(x, R, ub + T::SEQ[G][E] * CB_N, j, swj);
    cb_group_jobs<TK, G, E + 1>(x, xs, R, ub, j, swj);
  }
}

__device__ __forceinline__ void cb_cp_async16(cplx* smem_dst, const cplx* gsrc, bool valid) {   // zero fill when !valid
  const unsigned sa = (unsigned)__cvta_generic_to_shared(smem_dst);
  const int sz = valid ? 16 : 0;
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(sa), "l"(gsrc), "r"(sz) : "memory");
}

template <int TK>
__global__ void __launch_bounds__(CB_TH, 1) k_colb(ColbParams P) {
  constexpr int NSEQ = 2 * TK + 1;
  using PT = CbParts<TK>;
  using P1 = CbP1<TK>;
  constexpr int NACC = cb_max(cb_max(cb_part_pairs(PT::T0[0], PT::T1[0], PT::U0[0], PT::U1[0]),
                                     cb_part_pairs(PT::T0[1], PT::T1[1], PT::U0[1], PT::U1[1])),
                              cb_max(cb_part_pairs(PT::T0[2], PT::T1[2], PT::U0[2], PT::U1[2]), 1));
  constexpr int NPAIR = TK * (TK + 1) / 2 + TK;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx* sq = reinterpret_cast<cplx*>(smem_raw);   // [CB_G][NSEQ][CB_N]; phase 4: acs[NPAIR][CB_N]
  cplx* xstage = sq + CB_G * NSEQ * CB_N;         // [2 groups][8 blocks][CB_N]: staged second row images
  __shared__ cplx s_tw[CB_N];                     // e^{-2 pi i m/128}
  __shared__ int s_Dp[NPAIR];                     // lag half-range of every pair
  __shared__ cplx s_w[7 * 16];                    // w128^(j k1): row k1 - 1, lane j
  const int tid = threadIdx.x;
  const int H = P.H, D = P.D, B = P.B, nblk = P.nblk, nst = P.nst;
  const double invH = 1.0 / (double)H;
  const size_t imgStride = (size_t)(P.NC + 1) * H;      // T[img][y/G][kx][y%G] (k_row2_fwd)
  const size_t grpStride = (size_t)(P.NC + 1) * SFFT_T_G;
  for (int i = tid; i < CB_N; i += CB_TH) s_tw[i] = ldg2(P.tw128 + i);
  for (int i = tid; i < NPAIR; i += CB_TH) s_Dp[i] = P.pairs[i].D;
  for (int i = tid; i < 7 * 16; i += CB_TH) s_w[i] = ldg2(P.tw128 + ((i >> 4) + 1) * (i & 15));

  // phase-1 identity: warp = (group, block pair), half warp = block u of the stage, lane j
  const int p1_g = (tid >> 5) % 3, p1_u = ((tid >> 5) / 3) * 2 + ((tid >> 4) & 1), p1_j = tid & 15;
  constexpr int i00 = P1::IMG[0][0], i10 = P1::IMG[1][0], i20 = P1::IMG[2][0];
  constexpr int i01 = P1::IMG[0][1], i11 = P1::IMG[1][1], i21 = P1::IMG[2][1];
  const int p1_img0 = p1_g == 0 ? i00 : (p1_g == 1 ? i10 : i20);
  const int p1_img1 = p1_g == 0 ? i01 : (p1_g == 1 ? i11 : i21);
  const cplx* swj = s_w + p1_j;
  const int p2_k1 = tid & 7, p2_sub = tid >> 3;                        // phase 2
  const int p3_k = tid & (CB_N - 1), p3_part = tid >> 7;               // phase 3
  const int p3_pk = cb_slot(p3_k & 7, p3_k >> 3);

  // requests the 8 x 16 elements (n = j + 16 r) of block blk of row image img (zero past the block's end)
  auto fetch = [&](cplx* x, const cplx* Tcol, int blk, int img) {
    const int c0 = blk * B;
    const int lim = min(B, H - c0) + 2 * D;          // the last block may be short
    const cplx* src = Tcol + (size_t)img * imgStride;
    const int y0 = c0 - D + p1_j + H;
#pragma unroll
    for (int r = 0; r < 8; ++r) x[r] = (p1_j + 16 * r < lim) ? src[cb_toff((y0 + 16 * r) & (H - 1), grpStride)] : cmake(0.0, 0.0);
  };
  // the thread's inputs of stage st of column nkx: the group's first row image into registers (xa), its
  // second one (if any) by cp.async into the half warp's staging slot
  cplx xa[8];
  cplx* xs = xstage + ((p1_g > 0 ? p1_g - 1 : 0) * 8 + p1_u) * CB_N + p1_j;
  auto prefetch = [&](int nkx, int st) {
    if (nkx > P.NC) return;
    const int bs = (st * nblk) / nst, be = ((st + 1) * nblk) / nst;
    if (bs + p1_u >= be) return;
    const cplx* Tn = P.T + SFFT_T_G * (size_t)nkx;
    if (p1_img0 >= 0) fetch(xa, Tn, bs + p1_u, p1_img0);
    if (p1_img1 >= 0) {
      const int c0 = (bs + p1_u) * B;
      const int lim = min(B, H - c0) + 2 * D;
      const cplx* src = Tn + (size_t)p1_img1 * imgStride;
      const int y0 = c0 - D + p1_j + H;
#pragma unroll
      for (int r = 0; r < 8; ++r)
        cb_cp_async16(xs + 16 * r, src + cb_toff((y0 + 16 * r) & (H - 1), grpStride), p1_j + 16 * r < lim);
    }
    asm volatile("cp.async.commit_group;\n" ::: "memory");
  };
  prefetch(blockIdx.x, 0);
  __syncthreads();

  for (int kx = blockIdx.x; kx <= P.NC; kx += gridDim.x) {
    cplx acc[NACC];
#pragma unroll
    for (int i = 0; i < NACC; ++i) acc[i] = cmake(0.0, 0.0);

    for (int st = 0; st < nst; ++st) {
      const int b0 = (st * nblk) / nst, na = ((st + 1) * nblk) / nst - b0;     // blocks of this stage
      // ---- phase 1: weight, radix-8 over r (n = j + 16 r), twiddle, store ---------------------------
      if (p1_u < na) {
        const int c0 = (b0 + p1_u) * B;
        const int Bi = min(B, H - c0);
        const int Y = c0 - D + p1_j;             // unwrapped row of element r = 0
        CbRows R;
        R.e0 = (double)(2 * Y + 1 - H) * invH;
        R.step = 32.0 * invH;
        R.cenbits = R.lobits = R.hibits = 0u;
#pragma unroll
        for (int r = 0; r < 8; ++r) {
          const int n = p1_j + 16 * r;
          R.cenbits |= (n >= D && n < D + Bi) ? (1u << r) : 0u;
          R.lobits |= (Y + 16 * r < 0) ? (1u << r) : 0u;
          R.hibits |= (Y + 16 * r >= H) ? (1u << r) : 0u;
        }
        cplx* ub = sq + p1_u * NSEQ * CB_N;
        asm volatile("cp.async.wait_all;\n" ::: "memory");      // the lane's own staged elements have landed
        if (p1_g == 0) cb_group_jobs<TK, 0, 0>(xa, xs, R, ub, p1_j, swj);
        else if (p1_g == 1) cb_group_jobs<TK, 1, 0>(xa, xs, R, ub, p1_j, swj);
        else cb_group_jobs<TK, 2, 0>(xa, xs, R, ub, p1_j, swj);
      }
      __syncthreads();
      // ---- phase 2: radix-16 over j for every (block, sequence, k1) --------------------------------
      for (int it = p2_sub; it < na * NSEQ; it += CB_TH / 8) {
        cplx* sb = sq + it * CB_N + p2_k1 * 16;
        cplx v[16];
#pragma unroll
        for (int j = 0; j < 8; ++j) { v[j] = sb[j ^ p2_k1]; v[j + 8] = sb[(j ^ p2_k1) + 8]; }
        Dft<16, -1>::run(v);
#pragma unroll
        for (int k2 = 0; k2 < 8; ++k2) { sb[k2 ^ p2_k1] = v[k2]; sb[(k2 ^ p2_k1) + 8] = v[k2 + 8]; }   // X[k1 + 8 k2]
      }
      // the inputs of the thread's next stage (or of the next column's first stage) are requested now:
      // their latency hides under phase 3
      if (st + 1 < nst) prefetch(kx, st + 1);
      else prefetch(kx + gridDim.x, 0);
      __syncthreads();
      // ---- phase 3: products of the stage's blocks, accumulated in registers -----------------------
      for (int u = 0; u < na; ++u) {
        const cplx* ub = sq + u * NSEQ * CB_N;
        if (p3_part == 0) cb_accumulate<TK, PT::T0[0], PT::T1[0], PT::U0[0], PT::U1[0]>(acc, ub, p3_pk);
        else if (p3_part == 1) cb_accumulate<TK, PT::T0[1], PT::T1[1], PT::U0[1], PT::U1[1]>(acc, ub, p3_pk);
        else cb_accumulate<TK, PT::T0[2], PT::T1[2], PT::U0[2], PT::U1[2]>(acc, ub, p3_pk);
      }
      __syncthreads();
    }

    // ---- phase 4: accumulators -> lags ---------------------------------------------------------------
    cplx* acs = sq;
    if (p3_part == 0) cb_flush<TK, PT::T0[0], PT::T1[0], PT::U0[0], PT::U1[0]>(acc, acs, p3_k);
    else if (p3_part == 1) cb_flush<TK, PT::T0[1], PT::T1[1], PT::U0[1], PT::U1[1]>(acc, acs, p3_k);
    else cb_flush<TK, PT::T0[2], PT::T1[2], PT::U0[2], PT::U1[2]>(acc, acs, p3_k);
    __syncthreads();
    // (pair, a): V_a[m] = sum_b acs[a + 8 b] e^{+2 pi i b m/16}, in place (slot a + 8 m)
    {
      const int p4_a = tid & 7, p4_pair = tid >> 3;
      if (p4_pair < NPAIR) {     // NPAIR <= 27 < 48
        cplx V[16];
        cplx* base = acs + p4_pair * CB_N + p4_a;
#pragma unroll
        for (int b = 0; b < 16; ++b) V[b] = base[8 * b];
        Dft<16, +1>::run(V);
#pragma unroll
        for (int m = 0; m < 16; ++m) base[8 * m] = V[m];
      }
    }
    __syncthreads();
    // Y[dy] = (H/128) sum_a e^{+2 pi i a dy/128} V_a[dy mod 16]; the lanes start at different a (banks)
    const double scale = (double)H / (double)CB_N;
    for (int o = tid; o < NPAIR * CB_LAGS; o += CB_TH) {
      const int pair = o / CB_LAGS, dy = o - pair * CB_LAGS - 10;
      const int Dp = s_Dp[pair];
      if (dy < -Dp || dy > Dp) continue;
      const cplx* base = acs + pair * CB_N + 8 * ((dy + 16) & 15);
      cplx s = cmake(0.0, 0.0);
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        const int a = (i + tid) & 7;
        s = cadd(s, cmulc(s_tw[(a * (dy + 128)) & 127], base[a]));
      }
      P.Y[((size_t)pair * P.nLag + (dy + Dp)) * P.pitch + kx] = cscale(s, scale);
    }
    __syncthreads();   // the stage buffer is reused by the next column
  }
}

bool sfft_colx_supported(int H, int nPair) { return (H == 1024 || H == 2048 || H == 4096) && nPair <= 32; }

template <int TK>
static sfft_status launch_colb_t(const ColbParams& P, int num_sms, cudaStream_t st) {
  constexpr int NSEQ = 2 * TK + 1, NPAIR = TK * (TK + 1) / 2 + TK;
  const size_t smem = (size_t)(CB_G * NSEQ + 2 * 8) * CB_N * sizeof(cplx);   // stage buffer + staged second images
  static_assert((size_t)NPAIR * CB_N <= (size_t)CB_G * NSEQ * CB_N, "phase 4 scratch must fit the stage buffer");
  SFFT_CUDA_TRY(cudaFuncSetAttribute(k_colb<TK>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  int grid = num_sms;
  if (grid > P.NC + 1) grid = P.NC + 1;
  k_colb<TK><<<grid, CB_TH, smem, st>>>(P);
  SFFT_LAUNCH_CHECK();
  return SFFT_OK;
}

sfft_status sfft_launch_colx(sfft_plan* p, cudaStream_t st, int* nl) {
  ColbParams P;
  P.T = p->T; P.Y = p->Y; P.pairs = p->d_pairs; P.tw128 = p->tw128;
  P.H = p->H; P.NC = p->NC; P.pitch = p->pitch; P.nLag = p->nLag; P.nPair = p->nPair; P.nimg = p->nRowImg;
  P.D = p->Dmax; P.B = CB_N - 2 * p->Dmax; P.nblk = (p->H + P.B - 1) / P.B;
  P.nst = (P.nblk + CB_G - 1) / CB_G;
  ++*nl;
  switch (p->TK) {
    case 1: return launch_colb_t<1>(P, p->num_sms, st);
    case 3: return launch_colb_t<3>(P, p->num_sms, st);
    case 6: return launch_colb_t<6>(P, p->num_sms, st);
    default: return SFFT_ERR_UNSUPPORTED;
  }
}
