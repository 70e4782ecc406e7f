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
// One CTA per SM (persistent, columns round-robin), 512 threads in two roles that meet only at named
// barriers -- the transform warps never hold accumulators and the product warps never hold butterflies,
// which is what lets both stay inside 128 registers per thread:
//   producers (256 threads), per stage of CB_G blocks, into one of two shared-memory stage buffers:
//     phase 1  lanes (j < 16) x 16 groups: a group loads one row image's 8 x 16 block elements once and
//              produces that image's sequences one after the other: eta^q weighting, zero padding,
//              radix-8 butterflies over n = j + 16 r, twiddle w128^(j k1), store;
//     phase 2  radix-16 butterflies over j for every (block, sequence, k1): X[k1 + 8 k2];
//   consumers (256 threads), thread = (frequency k, half of the pairs):
//     phase 3  the stage's products accumulate in registers (9 operand loads per 13-14 pairs);
//     phase 4  (once per column, in the stage buffer it still owns) accumulators -> shared memory,
//              16-point inverse over b (k = a + 8 b), the 2D+1 lags of every pair, Y[pair][dy][kx].
// Shared-memory positions are XOR-swizzled (slot k1*16 + (j ^ k1)): every pass is conflict free with no
// padding.  T is column-major (T[img][kx][y]), so every load is a contiguous 256-byte run per half warp.
#include <math.h>
#include "fft_smem.cuh"

#define CB_N 128          // block transform length
#define CB_TH 512          // 256 producer + 256 consumer threads
#define CB_HALF 256
#define CB_G 4            // blocks per stage
#define CB_MAXTK 6        // DK <= 2
#define CB_MAXSUB 4       // sequences one phase-1 group produces
#define CB_LAGS 21        // 2 * 10 + 1

struct ColbParams {
  const cplx* T;          // [nimg][NC+1][H] column-major row spectra
  cplx* Y;                // [nPair][nLag][pitch]
  const PairDesc* pairs;
  const cplx* tw128;      // e^{-2 pi i m/128}, m < 128
  int H, NC, pitch, nLag, nPair, nimg;
  int D;                  // lag half-range (halo)
  int B;                  // centre rows per block = CB_N - 2 D
  int nblk;               // blocks per column = ceil(H / B)
  // phase-1 work table: group g < 4 of a block produces sub_n[g] sequences
  int sub_n[4];
  int sub_img[4][CB_MAXSUB], sub_q[4][CB_MAXSUB], sub_cen[4][CB_MAXSUB], sub_seq[4][CB_MAXSUB];
};

// pairs of half 0: centres t < TSPLIT, half 1: the rest (balanced for TK = 6: 13 / 14 pairs)
__host__ __device__ constexpr int cb_tsplit(int TK) { return TK == 6 ? 2 : (TK == 3 ? 1 : 1); }
__host__ __device__ constexpr int cb_npairs(int TK, int t0, int t1) {
  int n = 0;
  for (int t = t0; t < t1; ++t) n += TK - t + 1;   // (t, t..TK-1) and (t, S)
  return n;
}
__host__ __device__ constexpr int cb_max(int a, int b) { return a > b ? a : b; }

__device__ __forceinline__ int cb_slot(int k1, int j) { return k1 * 16 + (j ^ k1); }   // k1 < 8, j < 16

// Phase 3 for one block: acc[] += conj(C_t) E_t2 over the half's pairs, operands read once.
template <int TK, int T0, int T1>
__device__ __forceinline__ void cb_accumulate(cplx* acc, const cplx* __restrict__ ub, int pk) {
  cplx C[TK], E[TK + 1];
#pragma unroll
  for (int t = T0; t < T1; ++t) C[t] = ub[t * CB_N + pk];
#pragma unroll
  for (int t = T0; t <= TK; ++t) E[t] = ub[(TK + t) * CB_N + pk];
  int idx = 0;
#pragma unroll
  for (int t = T0; t < T1; ++t) {
#pragma unroll
    for (int t2 = t; t2 <= TK; ++t2) {
      cfmac(acc[idx], C[t], E[t2]);
      ++idx;
    }
  }
}

// Phase 4a: the half's accumulators -> shared memory acs[pair][k] (pair index of the plan's list:
// kernel-kernel pairs (t <= t2) row-major upper-triangular, then (t, S) at nKK + t)
template <int TK, int T0, int T1>
__device__ __forceinline__ void cb_flush(const cplx* acc, cplx* acs, int k) {
  constexpr int NKK = TK * (TK + 1) / 2;
  int idx = 0;
#pragma unroll
  for (int t = T0; t < T1; ++t) {
#pragma unroll
    for (int t2 = t; t2 <= TK; ++t2) {
      const int pair = (t2 < TK) ? (t * TK - t * (t - 1) / 2 + (t2 - t)) : (NKK + t);
      acs[pair * CB_N + k] = acc[idx];
      ++idx;
    }
  }
}

// named barriers (id 0 is __syncthreads)
#define CB_BAR_PROD 1      // producers, between phase 1 and phase 2
#define CB_BAR_CONS 2      // consumers, inside phase 4
#define CB_BAR_FULL 3      // +buffer: producers arrive, consumers wait
#define CB_BAR_EMPTY 5     // +buffer: consumers arrive, producers wait
__device__ __forceinline__ void cb_bar_sync(int id, int n) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory"); }
__device__ __forceinline__ void cb_bar_arrive(int id, int n) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(n) : "memory"); }

template <int TK>
__global__ void __launch_bounds__(CB_TH, 1) k_colb(ColbParams P) {
  constexpr int NSEQ = 2 * TK + 1;
  constexpr int TS = cb_tsplit(TK);
  constexpr int NACC = cb_max(cb_npairs(TK, 0, TS), cb_npairs(TK, TS, TK));
  constexpr int NPAIR = TK * (TK + 1) / 2 + TK;
  constexpr int STAGE = CB_G * NSEQ * CB_N;        // complex elements of one stage buffer
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx* sq = reinterpret_cast<cplx*>(smem_raw);   // [2][CB_G][NSEQ][CB_N]
  const int H = P.H, D = P.D, B = P.B, nblk = P.nblk;
  const int nst = (nblk + CB_G - 1) / CB_G;        // stages per column
  const int ncol = (P.NC + 1 - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;   // columns of this CTA
  const int total = ncol * nst;                    // stages of this CTA
  const size_t imgStride = (size_t)(P.NC + 1) * H;

  if (threadIdx.x < CB_HALF) {
    // =============================== producers ===================================================
    const int tid = threadIdx.x;
    const double invH = 1.0 / (double)H;
    const int p1_u = tid >> 6, p1_g = (tid >> 4) & 3, p1_j = tid & 15;
    const int p2_k1 = tid & 7, p2_sub = tid >> 3;
    const int ns = P.sub_n[p1_g];
    cplx tw[8];
#pragma unroll
    for (int k1 = 1; k1 < 8; ++k1) tw[k1] = ldg2(P.tw128 + p1_j * k1);   // j k1 <= 105
    int gs = 0;
    for (int kx = blockIdx.x; kx <= P.NC; kx += gridDim.x) {
      const cplx* Tcol = P.T + (size_t)kx * H;
      for (int b0 = 0; b0 < nblk; b0 += CB_G, ++gs) {
        cplx* buf = sq + (size_t)(gs & 1) * STAGE;
        if (gs >= 2) cb_bar_sync(CB_BAR_EMPTY + (gs & 1), CB_TH);   // the consumers are done with this buffer
        // ---- phase 1: load, weight, radix-8 over r (n = j + 16 r), twiddle, store ------------------
        const int blk = b0 + p1_u;
        if (blk < nblk && ns > 0) {
          const int c0 = blk * B;
          const int Bi = min(B, H - c0);        // the last block may be short
          int yr[8];
#pragma unroll
          for (int r = 0; r < 8; ++r) yr[r] = (c0 - D + p1_j + 16 * r + H) & (H - 1);
          cplx x[8];
          int cur = -1;
          cplx* ub = buf + (size_t)p1_u * NSEQ * CB_N;
          for (int s = 0; s < ns; ++s) {
            const int img = P.sub_img[p1_g][s], q = P.sub_q[p1_g][s];
            const bool wantCen = P.sub_cen[p1_g][s] != 0;
            if (img != cur) {
              const cplx* src = Tcol + (size_t)img * imgStride;
#pragma unroll
              for (int r = 0; r < 8; ++r) x[r] = (p1_j + 16 * r < Bi + 2 * D) ? __ldcs(src + yr[r]) : cmake(0.0, 0.0);
              cur = img;
            }
            cplx v[8];
#pragma unroll
            for (int r = 0; r < 8; ++r) {
              const int n = p1_j + 16 * r;
              const double eta = (double)(2 * yr[r] + 1 - H) * invH;
              double m = (q == 0) ? 1.0 : (q == 1 ? eta : eta * eta);
              if (wantCen && !(n >= D && n < D + Bi)) m = 0.0;
              v[r] = cscale(x[r], m);
            }
            Dft<8, -1>::run(v);
            cplx* dst = ub + (size_t)P.sub_seq[p1_g][s] * CB_N;
            dst[cb_slot(0, p1_j)] = v[0];
#pragma unroll
            for (int k1 = 1; k1 < 8; ++k1) dst[cb_slot(k1, p1_j)] = cmul(v[k1], tw[k1]);
          }
        }
        cb_bar_sync(CB_BAR_PROD, CB_HALF);
        // ---- phase 2: radix-16 over j for every (block, sequence, k1) ------------------------------
        const int nact = min(CB_G, nblk - b0) * NSEQ;
        for (int it = p2_sub; it < nact; it += CB_HALF / 8) {
          cplx* sb = buf + (size_t)it * CB_N + p2_k1 * 16;
          cplx v[16];
#pragma unroll
          for (int j = 0; j < 16; ++j) v[j] = sb[j ^ p2_k1];
          Dft<16, -1>::run(v);
#pragma unroll
          for (int k2 = 0; k2 < 16; ++k2) sb[k2 ^ p2_k1] = v[k2];   // X[k1 + 8 k2]
        }
        cb_bar_arrive(CB_BAR_FULL + (gs & 1), CB_TH);
      }
    }
  } else {
    // =============================== consumers ===================================================
    const int tid = threadIdx.x - CB_HALF;
    const int p3_k = tid & (CB_N - 1), p3_half = tid >> 7;
    const int p3_pk = cb_slot(p3_k & 7, p3_k >> 3);
    const double scale = (double)H / (double)CB_N;
    int gs = 0;
    for (int kx = blockIdx.x; kx <= P.NC; kx += gridDim.x) {
      cplx acc[NACC];
#pragma unroll
      for (int i = 0; i < NACC; ++i) acc[i] = cmake(0.0, 0.0);
      cplx* buf = sq;
      for (int b0 = 0; b0 < nblk; b0 += CB_G, ++gs) {
        buf = sq + (size_t)(gs & 1) * STAGE;
        cb_bar_sync(CB_BAR_FULL + (gs & 1), CB_TH);
        // ---- phase 3: products of the stage's blocks, accumulated in registers ---------------------
        const int na = min(CB_G, nblk - b0);
        for (int u = 0; u < na; ++u) {
          const cplx* ub = buf + (size_t)u * NSEQ * CB_N;
          if (p3_half == 0) cb_accumulate<TK, 0, TS>(acc, ub, p3_pk);
          else cb_accumulate<TK, TS, TK>(acc, ub, p3_pk);
        }
        // every stage but the column's last hands its buffer back at once
        if (b0 + CB_G < nblk && gs + 2 < total) cb_bar_arrive(CB_BAR_EMPTY + (gs & 1), CB_TH);
      }
      // ---- phase 4: accumulators -> lags, in the buffer of the column's last stage (still owned) ---
      cb_bar_sync(CB_BAR_CONS, CB_HALF);            // every consumer has finished reading the buffer
      cplx* acs = buf;
      if (p3_half == 0) cb_flush<TK, 0, TS>(acc, acs, p3_k);
      else cb_flush<TK, TS, TK>(acc, acs, p3_k);
      cb_bar_sync(CB_BAR_CONS, CB_HALF);
      // (pair, a): V_a[m] = sum_b acs[a + 8 b] e^{+2 pi i b m/16}, then w[pair][a][dy] = e^{2 pi i a dy/128} V_a[dy mod 16]
      cplx V[16];
      const int p4_a = tid & 7, p4_pair = tid >> 3;
      const bool p4_on = p4_pair < NPAIR;     // NPAIR <= 27 < 32
      if (p4_on) {
#pragma unroll
        for (int b = 0; b < 16; ++b) V[b] = acs[p4_pair * CB_N + p4_a + 8 * b];
        Dft<16, +1>::run(V);
      }
      cb_bar_sync(CB_BAR_CONS, CB_HALF);
      cplx* wr = buf;
      if (p4_on) {
#pragma unroll
        for (int i = 0; i < CB_LAGS; ++i) {
          const int dy = i - 10;
          if (dy >= -D && dy <= D) {
            const cplx t = ldg2(P.tw128 + ((p4_a * (dy + 128)) & 127));    // e^{-2 pi i a dy/128}
            wr[(p4_pair * 8 + p4_a) * CB_LAGS + i] = cmulc(t, V[(dy + 16) & 15]);
          }
        }
      }
      cb_bar_sync(CB_BAR_CONS, CB_HALF);
      for (int o = tid; o < NPAIR * CB_LAGS; o += CB_HALF) {
        const int pair = o / CB_LAGS, i = o - pair * CB_LAGS, dy = i - 10;
        const int Dp = P.pairs[pair].D;
        if (dy < -Dp || dy > Dp) continue;
        cplx s = cmake(0.0, 0.0);
#pragma unroll
        for (int a = 0; a < 8; ++a) s = cadd(s, wr[(pair * 8 + a) * CB_LAGS + i]);
        P.Y[((size_t)pair * P.nLag + (dy + Dp)) * P.pitch + kx] = cscale(s, scale);
      }
      // the column's last stage buffer goes back to the producers (unless nobody will wait for it)
      if (gs - 1 + 2 < total) cb_bar_arrive(CB_BAR_EMPTY + ((gs - 1) & 1), CB_TH);
    }
  }
}

bool sfft_colx_supported(int H, int nPair) { return (H == 1024 || H == 2048 || H == 4096) && nPair <= 32; }

template <int TK>
static sfft_status launch_colb_t(const ColbParams& P, int num_sms, cudaStream_t st) {
  constexpr int NSEQ = 2 * TK + 1, NPAIR = TK * (TK + 1) / 2 + TK;
  const size_t stage = (size_t)CB_G * NSEQ * CB_N * sizeof(cplx);
  static_assert((size_t)cb_max(NPAIR * CB_N, NPAIR * 8 * CB_LAGS) <= (size_t)CB_G * NSEQ * CB_N,
                "phase 4 scratch must fit one stage buffer");
  const size_t smem = 2 * stage;
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
  // phase-1 work table.  Sequence index: centre of monomial t at t, extended at TK + t, S~ at 2 TK.
  // The sequences of one row image are packed into groups of <= CB_MAXSUB so that a group reads its
  // image once; the four groups of a block are filled greedily, largest image first.
  struct Seq { int img, q, cen, seq; };
  Seq all[2 * CB_MAXTK + 1];
  int n = 0;
  const int TK = p->TK;
  for (int cen = 0; cen < 2; ++cen)
    for (int t = 0; t < TK; ++t) {
      all[n].img = p->monoK[t][0]; all[n].q = p->monoK[t][1]; all[n].cen = cen; all[n].seq = cen ? t : TK + t; ++n;
    }
  all[n].img = p->DK + 1; all[n].q = 0; all[n].cen = 0; all[n].seq = 2 * TK; ++n;
  for (int g = 0; g < 4; ++g) P.sub_n[g] = 0;
  // chunks: (image, extended/centre) lists in image order
  for (int img = 0; img <= p->DK + 1; ++img)
    for (int cen = 0; cen < 2; ++cen) {
      // the least loaded group that has room takes this chunk (chunks of one image share the load)
      int cnt = 0;
      for (int i = 0; i < n; ++i) cnt += (all[i].img == img && all[i].cen == cen);
      if (!cnt) continue;
      int best = -1;
      for (int g = 0; g < 4; ++g)
        if (P.sub_n[g] + cnt <= CB_MAXSUB && (best < 0 || P.sub_n[g] < P.sub_n[best])) best = g;
      if (best < 0) return SFFT_ERR_UNSUPPORTED;
      for (int i = 0; i < n; ++i)
        if (all[i].img == img && all[i].cen == cen) {
          const int k = P.sub_n[best]++;
          P.sub_img[best][k] = all[i].img; P.sub_q[best][k] = all[i].q;
          P.sub_cen[best][k] = all[i].cen; P.sub_seq[best][k] = all[i].seq;
        }
    }
  ++*nl;
  switch (TK) {
    case 1: return launch_colb_t<1>(P, p->num_sms, st);
    case 3: return launch_colb_t<3>(P, p->num_sms, st);
    case 6: return launch_colb_t<6>(P, p->num_sms, st);
    default: return SFFT_ERR_UNSUPPORTED;
  }
}
