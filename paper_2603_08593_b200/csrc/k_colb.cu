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
// 2D+1 twiddled accumulations per 8 frequencies) this needs 1.5x fewer fp64 operations at the full
// CCD, and a quarter of them are plain complex multiply-accumulates.  The sequences are the column kx
// of the row spectra T (k_row2_fwd), f = eta^q T_p for every kernel monomial t = (p,q) ("centre" AND
// "extended" version: 2 TK sequences) and g = the row spectrum of m S ("extended" only).
//
// One persistent CTA per SM (columns round-robin), 16 warps in two ROLES that meet only at mbarriers (no
// block-wide barrier after the prologue); registers are rebalanced between the warpgroups with setmaxnreg:
//   transform warps (12, 120 registers)  run "tasks" of four sequences, warp-synchronously: each half warp
//            (lane j < 16) takes the 8 x 16 block elements n = j + 16 r of its row image from global memory
//            (requested one task ahead: CB_PREG in registers, the rest by cp.async, issued after the
//            radix-16 pass has issued its shared-memory loads), and per sequence weights them by eta^q,
//            zero-pads (centre version), runs the radix-8 butterfly over r, multiplies by w128^(j k1) and
//            stores to the block's slot of the shared-memory ring; after a __syncwarp the 32 lanes run the
//            radix-16 butterflies over j of the four sequences (X[k1 + 8 k2]) in place, and lane 0 arrives
//            on the slot's "full" barrier.  Task g of the CTA's task list (all its columns, block by block)
//            runs on warp g mod 12.  The science sequence (one per block) is batched over four consecutive
//            blocks into a task of its own and goes to a ring of its own (CB_NS2 blocks), so that it never
//            waits for the main ring;
//   product warps (4, 152 registers)  thread = frequency k; they wait for a slot to be full, read each of its
//            2TK+1 spectra ONCE and accumulate all TK(TK+1)/2 + TK pair products conj(C_t) E_t2 in registers
//            over the blocks of a column, then free the slot ("empty" barrier).  End of a column:
//            accumulators -> shared memory (two passes over half of the pairs), 16-point inverse over b
//            (k = a + 8 b), the 2D+1 lags of every pair (8 twiddled terms each) -> Y[pair][dy][kx].
// The ring holds CB_NSLOT blocks, so the transforms run up to CB_NSLOT blocks ahead of the products, also
// across the column boundary; both roles issue to the same fp64 pipes at the same time.
// Shared-memory positions are XOR-swizzled (slot k1*16 + (j ^ k1)): every pass is conflict free with no
// padding.  T has the row-group layout T[img][y/G][kx][y%G], G = SFFT_T_G = 4 (k_row2_fwd): a half warp's
// 16 rows of a column are four 64-byte runs.
#include <math.h>
#include "fft_smem.cuh"

#define CB_N 128          // block transform length
#define CB_TH 512         // 16 warps = 4 warpgroups: 3 transform + 1 product (registers rebalanced by setmaxnreg)
#define CB_FW 12          // transform warps
#ifndef CB_PREG
#define CB_PREG 5           // block elements (of 8) a transform lane prefetches into registers (the rest: cp.async)
#endif
#define CB_REG_F 120       // registers per thread of the transform warpgroups
#define CB_REG_P 152       // ... of the product warpgroup (3 x 120 + 152 = 4 x 128)
#define CB_PT 128         // product threads (one per frequency)
#ifndef CB_NSLOT
#define CB_NSLOT 6        // blocks in the shared-memory ring
#endif
#ifndef CB_NS2
#define CB_NS2 16         // blocks in the ring of the S~ spectra (DK = 2: they are produced four blocks at a time, ahead of the rest)
#endif
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
};

// ---- task tables ---------------------------------------------------------------------------------------
// Sequence index inside a slot: centre version of monomial t at t, extended version at TK + t, S~
// (extended only) at 2 TK.  Monomial order (p,q): DK = 2: (0,0),(1,0),(0,1),(2,0),(1,1),(0,2); DK = 1:
// (0,0),(1,0),(0,1); row image = p (S~ is image DK + 1), q = power of eta.
// A per-block task = 2 half warps x 2 jobs; a half warp reads ONE row image.  Descriptor of a half warp:
//   bits 0-1 image | job 0: bits 2-3 q, bit 4 centre, bits 5-8 sequence, bit 9 valid | job 1: the same at 10-17.
// Where the images allow it the two half warps of a job share q (no divergence on the weighting branch).
__host__ __device__ constexpr unsigned cb_job(int q, int cen, int seq) { return (unsigned)(q | (cen << 2) | (seq << 3) | (1 << 7)); }
__host__ __device__ constexpr unsigned cb_half(int img, unsigned j0, unsigned j1) { return (unsigned)img | (j0 << 2) | (j1 << 10); }
template <int TK> struct CbTasks;
template <> struct CbTasks<6> {
  static constexpr int NT = 3;            // tasks per block
  static constexpr bool STASK = true;     // S~ sequences: a task of their own over 4 consecutive blocks
  static constexpr int SIMG = 3, SSEQ = 12;
  __device__ static constexpr unsigned desc(int task, int half) {
    return task == 0 ? (half == 0 ? cb_half(0, cb_job(0, 0, 6), cb_job(1, 0, 8))      // E(0,0) E(0,1)
                                  : cb_half(0, cb_job(0, 1, 0), cb_job(1, 1, 2)))     // C(0,0) C(0,1)
         : task == 1 ? (half == 0 ? cb_half(1, cb_job(0, 0, 7), cb_job(1, 0, 10))     // E(1,0) E(1,1)
                                  : cb_half(1, cb_job(0, 1, 1), cb_job(1, 1, 4)))     // C(1,0) C(1,1)
                     : (half == 0 ? cb_half(2, cb_job(0, 0, 9), cb_job(0, 1, 3))      // E(2,0) C(2,0)
                                  : cb_half(0, cb_job(2, 0, 11), cb_job(2, 1, 5)));   // E(0,2) C(0,2)
  }
};
template <> struct CbTasks<3> {
  static constexpr int NT = 2;
  static constexpr bool STASK = false;
  static constexpr int SIMG = 2, SSEQ = 6;
  __device__ static constexpr unsigned desc(int task, int half) {
    return task == 0 ? (half == 0 ? cb_half(0, cb_job(0, 0, 3), cb_job(1, 0, 5))      // E(0,0) E(0,1)
                                  : cb_half(0, cb_job(0, 1, 0), cb_job(1, 1, 2)))     // C(0,0) C(0,1)
                     : (half == 0 ? cb_half(1, cb_job(0, 0, 4), cb_job(0, 1, 1))      // E(1,0) C(1,0)
                                  : cb_half(2, cb_job(0, 0, 6), 0u));                 // S~
  }
};
template <> struct CbTasks<1> {
  static constexpr int NT = 1;
  static constexpr bool STASK = false;
  static constexpr int SIMG = 1, SSEQ = 2;
  __device__ static constexpr unsigned desc(int task, int half) {
    return half == 0 ? cb_half(0, cb_job(0, 0, 1), cb_job(0, 1, 0))                   // E(0,0) C(0,0)
                     : cb_half(1, cb_job(0, 0, 2), 0u);                               // S~
  }
};

__device__ __forceinline__ int cb_slot(int k1, int j) { return k1 * 16 + (j ^ k1); }   // k1 < 8, j < 16

// offset of row y inside one image of T (column 0): T[img][y/G][kx][y%G], G = SFFT_T_G
__device__ __forceinline__ size_t cb_toff(int y, size_t grpStride) {
  return (size_t)(y / SFFT_T_G) * grpStride + (size_t)(y % SFFT_T_G);
}

// ---- mbarrier helpers (CTA scope; `a` = 32-bit shared-memory address of the barrier) -------------------
__device__ __forceinline__ unsigned smem_addr(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned a, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(a), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned a) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" ::"r"(a) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned a, unsigned parity) {
  unsigned done;
  do {
    asm volatile(
        "{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}\n"
        : "=r"(done) : "r"(a), "r"(parity) : "memory");
  } while (!done);
}
__device__ __forceinline__ void cb_bar_products() {   // the 128 product threads only
  asm volatile("bar.sync 1, %0;\n" ::"n"(CB_PT) : "memory");
}

// One phase-1 job of a half warp: sequence = DFT8 over r of (x[r] * eta_r^q, zero outside the centre rows
// when cen), twiddled by w128^(j k1) (w^1, w^2 from s_w, lane j; higher powers as products) and stored at the lane's positions
// of `dst`.  q and cen are uniform over a half warp.  e0 = eta of the lane's element r = 0 (unwrapped row),
// estep = 32/H; edge: the block is the first or one of the last two of its column (rows may wrap, the centre may be
// short), Yrow = unwrapped row of element 0, Bi = the block's centre rows.
__device__ __forceinline__ void cb_job_run(const cplx* x, int q, bool cen, cplx* dst, int j, const cplx* __restrict__ swj,
                                           double e0, double estep, bool edge, int Yrow, int Bi, int D, int H) {
  cplx v[8];
#pragma unroll
  for (int r = 0; r < 8; ++r) v[r] = x[r];
  if (q > 0) {
#pragma unroll
    for (int r = 0; r < 8; ++r) {
      double e = fma((double)r, estep, e0);
      if (edge) {                         // every value is a multiple of 1/H: exact
        if (Yrow + 16 * r < 0) e += 2.0;
        if (Yrow + 16 * r >= H) e -= 2.0;
      }
      if (q == 2) e *= e;
      v[r] = cscale(v[r], e);
    }
  }
  if (cen) {
    // centre rows: n = j + 16 r in [D, D + Bi); with D <= 16 only r = 0 (and r = 7 for a whole block) can fall outside
    if (j < D) v[0] = cmake(0.0, 0.0);
    if (!edge) {
      if (j + 112 >= D + Bi) v[7] = cmake(0.0, 0.0);
    } else {
      // (r = 0 included: the last block of a column can hold fewer than 16 - D centre rows, e.g. H = 2048, w = 2)
#pragma unroll
      for (int r = 0; r < 8; ++r)
        if (j + 16 * r >= D + Bi) v[r] = cmake(0.0, 0.0);
    }
  }
  Dft<8, -1>::run(v);
  dst[cb_slot(0, j)] = v[0];
#pragma unroll
  {  // w^k1, w = w128^j: w^1 and w^2 from the table, the rest as products (depth <= 2): 5 fewer shared loads per job
     // (0.280 -> 0.278 ms per launch; the kernel is co-limited by the shared-memory pipe)
    const cplx w1 = swj[0], w2 = swj[16];
    const cplx w3 = cmul(w1, w2), w4 = csqr(w2);
    dst[cb_slot(1, j)] = cmul(v[1], w1);
    dst[cb_slot(2, j)] = cmul(v[2], w2);
    dst[cb_slot(3, j)] = cmul(v[3], w3);
    dst[cb_slot(4, j)] = cmul(v[4], w4);
    dst[cb_slot(5, j)] = cmul(v[5], cmul(w1, w4));
    dst[cb_slot(6, j)] = cmul(v[6], cmul(w2, w4));
    dst[cb_slot(7, j)] = cmul(v[7], cmul(w3, w4));
  }
}

template <int TK>
__global__ void __launch_bounds__(CB_TH, 1) k_colb(ColbParams P) {
  constexpr int NSEQ = 2 * TK + 1;
  constexpr int NPAIR = TK * (TK + 1) / 2 + TK;
  using TT = CbTasks<TK>;
  constexpr unsigned FULL_COUNT = TT::NT;                         // lane-0 arrivals that complete a block
  constexpr int NGRP_T = TT::STASK ? (1 + 4 * TT::NT) : TT::NT;   // tasks of a group of 4 blocks (or of one block)
  constexpr int NSEQ_R = TT::STASK ? NSEQ - 1 : NSEQ;             // sequences per slot of the main ring
  constexpr int SRING = CB_NSLOT * NSEQ_R * CB_N;                 // element offset of the S~ ring
  constexpr int NPASS4 = NPAIR > 16 ? 2 : 1;                      // the end-of-column inverse runs in NPASS4 passes
  constexpr int PP4 = (NPAIR + NPASS4 - 1) / NPASS4;              // over PP4 pairs each (scratch size)
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx* ring = reinterpret_cast<cplx*>(smem_raw);        // [CB_NSLOT][NSEQ_R][CB_N], then [CB_NS2][CB_N] (S~ ring)
  cplx* acs = ring + SRING + (TT::STASK ? CB_NS2 * CB_N : 0);   // [PP4][CB_N]: end-of-column scratch
  __shared__ cplx s_tw[CB_N];                            // e^{-2 pi i m/128}
  __shared__ cplx s_w[2 * 16];                           // w128^(j k1), k1 = 1, 2: row k1 - 1, lane j
  __shared__ int s_Dp[NPAIR];                            // lag half-range of every pair
  __shared__ cplx s_xs[(8 - CB_PREG) * CB_FW * 32];      // a transform lane's prefetched elements r >= CB_PREG (cp.async)
  __shared__ __align__(8) unsigned long long s_full[CB_NSLOT], s_empty[CB_NSLOT], s_sfull[CB_NS2], s_sempty[CB_NS2];
  const int tid = threadIdx.x, lane = tid & 31, wrp = tid >> 5;
  const int H = P.H, D = P.D, B = P.B, nblk = P.nblk;
  const double invH = 1.0 / (double)H, estep = 32.0 * invH;
  const size_t imgStride = (size_t)(P.NC + 1) * H;       // T[img][y/G][kx][y%G] (k_row2_fwd)
  const unsigned grpStride = (unsigned)(P.NC + 1) * SFFT_T_G;
  for (int i = tid; i < CB_N; i += CB_TH) s_tw[i] = ldg2(P.tw128 + i);
  for (int i = tid; i < 2 * 16; i += CB_TH) s_w[i] = ldg2(P.tw128 + ((i >> 4) + 1) * (i & 15));
  for (int i = tid; i < NPAIR; i += CB_TH) s_Dp[i] = P.pairs[i].D;
  // 32-bit shared addresses of the barrier arrays (barrier i at base + 8 i)
  const unsigned aFull = smem_addr(s_full), aEmpty = smem_addr(s_empty), aSFull = smem_addr(s_sfull), aSEmpty = smem_addr(s_sempty);
  if (tid < CB_NSLOT) {
    mbar_init(aFull + 8u * tid, FULL_COUNT);
    mbar_init(aEmpty + 8u * tid, CB_PT / 32);
  }
  if (tid < CB_NS2) {
    mbar_init(aSFull + 8u * tid, 1);
    mbar_init(aSEmpty + 8u * tid, CB_PT / 32);
  }
  __syncthreads();
  const int ncolMine = (P.NC + 1 - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;   // columns of this CTA

  // ---- transform side: the warp's task cursor (ti = task index inside column iteration tci)
  const int half = lane >> 4, j = lane & 15;
  const cplx* swj = s_w + j;
  const int tasksPerCol = TT::STASK ? (TT::NT * nblk + (nblk + 3) / 4) : TT::NT * nblk;
  // A warp's consecutive tasks must lie at most one ring generation (CB_NSLOT blocks) apart: the parity wait on
  // an empty-barrier only tells the previous generation from the current one.  With one task per block (TK = 1)
  // twelve warps would span two generations, so only FWA of them take tasks there (the others idle).
  constexpr int FWA = TT::STASK ? CB_FW : (CB_FW < TT::NT * CB_NSLOT ? CB_FW : TT::NT * CB_NSLOT);
  int tci = wrp < FWA ? 0 : ncolMine, ti = wrp;   // (transform warps only)
  while (ti >= tasksPerCol && tci < ncolMine) { ti -= tasksPerCol; ++tci; }
  // decode ti -> (type, first block); type < NT: per-block task, type == NT: S~ task over blocks blk .. blk + 3
  auto decode = [&](int lid, int& type, int& blk) {
    if (TT::STASK) {
      const int m = lid / NGRP_T, rem = lid - m * NGRP_T;
      if (rem == 0) { type = TT::NT; blk = 4 * m; }
      else { type = (rem - 1) % TT::NT; blk = 4 * m + (rem - 1) / TT::NT; }
    } else {
      type = lid % TT::NT; blk = lid / TT::NT;
    }
  };
  auto lane_img = [&](int type) -> int { return type == TT::NT ? TT::SIMG : (int)(TT::desc(type, half) & 3u); };
  auto job_blk = [&](int type, int blk, int jb) -> int { return type == TT::NT ? blk + 2 * half + jb : blk; };
  // requests the 8 x 16 elements (n = j + 16 r) of block b of row image img, column kx (zero past the block's end)
  // (elements r in [R0, R1): the prefetch of a task is issued in two parts, see run_task)
  auto fetch = [&](cplx* x, int kx, int b, int img, int R0 = 0, int R1 = 8) {
    const int c0 = b * B;
    const int lim = b < nblk ? min(B, H - c0) + 2 * D : 0;   // the last block may be short
    const cplx* src = P.T + SFFT_T_G * (size_t)kx + (size_t)img * imgStride;
    const int y0 = (c0 - D + j + H) & (H - 1);               // row of element r = 0; rows r differ by 16 = 2 groups
    const unsigned gi0 = (unsigned)y0 / SFFT_T_G, sub = (unsigned)y0 % SFFT_T_G, gmask = (unsigned)(H / SFFT_T_G) - 1u;
#pragma unroll
    for (int r = R0; r < R1; ++r) {
      const unsigned gi = (gi0 + (unsigned)(16 / SFFT_T_G) * r) & gmask;
      x[r] = (j + 16 * r < lim) ? src[gi * grpStride + sub] : cmake(0.0, 0.0);
    }
  };
  // prefetch of a task's first job: elements r < CB_PREG into registers, the others by cp.async into the
  // lane's staging words (the radix-16 pass that runs meanwhile needs the registers); prefetch_land()
  // completes it
  const unsigned aStage = smem_addr(&s_xs[tid < CB_FW * 32 ? tid : 0]);   // the lane's staging words, CB_FW*32*16 bytes apart
  auto prefetch = [&](cplx* x, int kx, int b, int img) {
    fetch(x, kx, b, img, 0, CB_PREG);
    const int c0 = b * B;
    const int lim = b < nblk ? min(B, H - c0) + 2 * D : 0;
    const cplx* src = P.T + SFFT_T_G * (size_t)kx + (size_t)img * imgStride;
    const int y0 = (c0 - D + j + H) & (H - 1);
    const unsigned gi0 = (unsigned)y0 / SFFT_T_G, sub = (unsigned)y0 % SFFT_T_G, gmask = (unsigned)(H / SFFT_T_G) - 1u;
#pragma unroll
    for (int r = CB_PREG; r < 8; ++r) {
      const unsigned gi = (gi0 + (unsigned)(16 / SFFT_T_G) * r) & gmask;
      const bool in = j + 16 * r < lim;
      const int sz = in ? 16 : 0;                           // zero fill past the block's end
      asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n"
                   ::"r"(aStage + (unsigned)((r - CB_PREG) * CB_FW * 32 * sizeof(cplx))), "l"(src + (in ? gi * grpStride + sub : 0u)), "r"(sz) : "memory");
    }
    asm volatile("cp.async.commit_group;\n" ::: "memory");
  };
  auto prefetch_land = [&](cplx* x) {
    asm volatile("cp.async.wait_all;\n" ::: "memory");
#pragma unroll
    for (int r = CB_PREG; r < 8; ++r) x[r] = s_xs[(r - CB_PREG) * CB_FW * 32 + tid];
  };
  cplx xa[8];
  int ttype = 0, tblk = 0;
  if (tci < ncolMine && wrp < CB_FW) {
    decode(ti, ttype, tblk);
    prefetch(xa, (int)blockIdx.x + tci * (int)gridDim.x, job_blk(ttype, tblk, 0), lane_img(ttype));
  }
  auto run_task = [&]() {
    const int kx = (int)blockIdx.x + tci * (int)gridDim.x;
    const int nbase = tci * nblk;
    const bool stask = TT::STASK && ttype == TT::NT;
    const unsigned desc = stask ? cb_half(TT::SIMG, cb_job(0, 0, TT::SSEQ), cb_job(0, 0, TT::SSEQ)) : TT::desc(ttype, half);
    prefetch_land(xa);
    // ---- phase 1: two jobs per half warp
    int soff[2];        // element offset of the job's sequence in the ring, -1 = no job
#pragma unroll
    for (int jb = 0; jb < 2; ++jb) {
      const unsigned jd = (desc >> (2 + 8 * jb)) & 0xffu;
      const int b = job_blk(ttype, tblk, jb);
      const bool valid = ((jd >> 7) & 1u) && b < nblk;
      soff[jb] = !valid ? -1 : stask ? SRING + ((nbase + b) % CB_NS2) * CB_N
                                     : (((nbase + b) % CB_NSLOT) * NSEQ_R + (int)((jd >> 3) & 15u)) * CB_N;
      if (stask && jb == 1) fetch(xa, kx, b, TT::SIMG);   // the S~ task reads a new block per job
      if (valid) {
        const int c0 = b * B, Yrow = c0 - D + j;
        cb_job_run(xa, (int)(jd & 3u), ((jd >> 2) & 1u) != 0u, ring + soff[jb], j, swj,
                   (double)(2 * Yrow + 1 - H) * invH, estep, b == 0 || b >= nblk - 2, Yrow, min(B, H - c0), D, H);
      }
    }
    // ---- advance the cursor; the next task's inputs are requested now (their latency hides under phase 2,
    //      the products and the waits)
    const int pblk = tblk;
    ti += FWA;
    while (ti >= tasksPerCol && tci < ncolMine) { ti -= tasksPerCol; ++tci; }
    if (tci < ncolMine) decode(ti, ttype, tblk);
    __syncwarp();
    // ---- phase 2: radix-16 over j; lane = (sequence sq = (half, job), k1)
    {
      const int sq = lane >> 3, k1 = lane & 7;
      const int o0 = __shfl_sync(0xffffffffu, soff[0], (sq >> 1) * 16), o1 = __shfl_sync(0xffffffffu, soff[1], (sq >> 1) * 16);
      const int off = (sq & 1) ? o1 : o0;
      cplx* base = ring + (off >= 0 ? off : 0) + k1 * 16;
      cplx v[16];   // (a lane without a sequence transforms slot 0 and stores nothing)
#pragma unroll
      for (int jj = 0; jj < 8; ++jj) { v[jj] = base[jj ^ k1]; v[jj + 8] = base[(jj ^ k1) + 8]; }
      // the next task's inputs are requested HERE, after the shared-memory loads of this pass have been
      // issued (issued earlier, the global loads' scoreboard would hold up those loads and the shuffles):
      // their latency hides under the butterfly, the stores and the waits that follow
      asm volatile("" ::: "memory");
      if (tci < ncolMine) prefetch(xa, (int)blockIdx.x + tci * (int)gridDim.x, job_blk(ttype, tblk, 0), lane_img(ttype));
      asm volatile("" ::: "memory");
      Dft<16, -1>::run(v);
      if (off >= 0) {
#pragma unroll
        for (int k2 = 0; k2 < 8; ++k2) { base[k2 ^ k1] = v[k2]; base[(k2 ^ k1) + 8] = v[k2 + 8]; }   // X[k1 + 8 k2]
      }
    }
    __syncwarp();
    if (lane == 0) {
      if (stask) {
#pragma unroll
        for (int i = 0; i < 4; ++i)
          if (pblk + i < nblk) mbar_arrive(aSFull + 8u * (unsigned)((nbase + pblk + i) % CB_NS2));
      } else {
        mbar_arrive(aFull + 8u * (unsigned)((nbase + pblk) % CB_NSLOT));
      }
    }
  };

  if (wrp < CB_FW) {
    // =============================== transform warps ===============================================
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;\n" ::"n"(CB_REG_F));
    while (tci < ncolMine) {
      const int nb = tci * nblk + tblk;
      if (TT::STASK && ttype == TT::NT) {
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          const int n = nb + i;
          if (tblk + i < nblk) mbar_wait(aSEmpty + 8u * (unsigned)(n % CB_NS2), (unsigned)(((n / CB_NS2) & 1) ^ 1));
        }
      } else {
        mbar_wait(aEmpty + 8u * (unsigned)(nb % CB_NSLOT), (unsigned)(((nb / CB_NSLOT) & 1) ^ 1));
      }
      run_task();
    }
  } else {
    // =============================== product warps ================================================
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;\n" ::"n"(CB_REG_P));
    constexpr int NKK = TK * (TK + 1) / 2;
    const int k = tid - CB_FW * 32;                      // frequency
    const int pk = cb_slot(k & 7, k >> 3);
    const double scale = (double)H / (double)CB_N;
    int n = 0;                                           // block sequence number
    for (int ci = 0; ci < ncolMine; ++ci) {
      const int kx = (int)blockIdx.x + ci * (int)gridDim.x;
      cplx acc[NPAIR];
#pragma unroll
      for (int i = 0; i < NPAIR; ++i) acc[i] = cmake(0.0, 0.0);
      for (int b = 0; b < nblk; ++b, ++n) {
        const int slot = n % CB_NSLOT;
        mbar_wait(aFull + 8u * (unsigned)slot, (unsigned)((n / CB_NSLOT) & 1));
        if (TT::STASK) mbar_wait(aSFull + 8u * (unsigned)(n % CB_NS2), (unsigned)((n / CB_NS2) & 1));
        const cplx* ub = ring + (size_t)slot * NSEQ_R * CB_N + pk;
        const cplx* us = TT::STASK ? ring + SRING + (n % CB_NS2) * CB_N + pk : ub + 2 * TK * CB_N;
        cplx C[TK];
#pragma unroll
        for (int t = 0; t < TK; ++t) C[t] = ub[t * CB_N];
#pragma unroll
        for (int t2 = 0; t2 <= TK; ++t2) {
          const cplx E = t2 < TK ? ub[(TK + t2) * CB_N] : us[0];
#pragma unroll
          for (int t = 0; t < TK; ++t) {
            if (t <= t2) {
              const int pair = (t2 < TK) ? (t * TK - t * (t - 1) / 2 + (t2 - t)) : (NKK + t);
              cfmac(acc[pair], C[t], E);
            }
          }
        }
        __syncwarp();
        if (lane == 0) {
          mbar_arrive(aEmpty + 8u * (unsigned)slot);
          if (TT::STASK) mbar_arrive(aSEmpty + 8u * (unsigned)(n % CB_NS2));
        }
      }
      // ---- end of the column: accumulators -> lags, PP4 pairs at a time
#pragma unroll
      for (int ps = 0; ps < NPASS4; ++ps) {
        const int p0 = ps * PP4, np = (NPAIR - p0 < PP4) ? NPAIR - p0 : PP4;
#pragma unroll
        for (int i = 0; i < NPAIR; ++i)
          if (i >= p0 && i < p0 + PP4) acs[(i - p0) * CB_N + k] = acc[i];
        cb_bar_products();
        // (pair, a): V_a[m] = sum_b acs[a + 8 b] e^{+2 pi i b m/16}, in place (position a + 8 m)
        for (int it = k; it < np * 8; it += CB_PT) {
          const int a = it & 7, pl = it >> 3;
          cplx V[16];
          cplx* base = acs + pl * CB_N + a;
#pragma unroll
          for (int bb = 0; bb < 16; ++bb) V[bb] = base[8 * bb];
          Dft<16, +1>::run(V);
#pragma unroll
          for (int m = 0; m < 16; ++m) base[8 * m] = V[m];
        }
        cb_bar_products();
        // Y[dy] = (H/128) sum_a e^{+2 pi i a dy/128} V_a[dy mod 16]; the lanes start at different a (banks)
        for (int o = k; o < np * CB_LAGS; o += CB_PT) {
          const int pl = o / CB_LAGS, dy = o - pl * CB_LAGS - 10, pair = p0 + pl;
          const int Dp = s_Dp[pair];
          if (dy < -Dp || dy > Dp) continue;
          const cplx* base = acs + pl * CB_N + 8 * ((dy + 16) & 15);
          cplx s = cmake(0.0, 0.0);
#pragma unroll
          for (int i = 0; i < 8; ++i) {
            const int a = (i + k) & 7;
            s = cadd(s, cmulc(s_tw[(a * (dy + 128)) & 127], base[a]));
          }
          P.Y[((size_t)pair * P.nLag + (dy + Dp)) * P.pitch + kx] = cscale(s, scale);
        }
        cb_bar_products();   // the scratch is rewritten by the next pass / at the end of the next column
      }
    }
  }
}

// (lag half-ranges above 10, i.e. w > 5, take the generic column and cross kernels)
bool sfft_colx_supported(int H, int nPair, int Dmax) { return (H == 1024 || H == 2048 || H == 4096) && nPair <= 32 && Dmax <= 10; }

template <int TK>
static sfft_status launch_colb_t(const ColbParams& P, int num_sms, cudaStream_t st) {
  constexpr int NSEQ = 2 * TK + 1, NPAIR = TK * (TK + 1) / 2 + TK;
  constexpr bool ST = CbTasks<TK>::STASK;
  constexpr int NP4 = NPAIR > 16 ? 2 : 1, PP4 = (NPAIR + NP4 - 1) / NP4;
  // ring (+ S~ ring) + end-of-column scratch
  const size_t smem = (size_t)(CB_NSLOT * (ST ? NSEQ - 1 : NSEQ) + (ST ? CB_NS2 : 0) + PP4) * CB_N * sizeof(cplx);
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
  ++*nl;
  switch (p->TK) {
    case 1: return launch_colb_t<1>(P, p->num_sms, st);
    case 3: return launch_colb_t<3>(P, p->num_sms, st);
    case 6: return launch_colb_t<6>(P, p->num_sms, st);
    default: return SFFT_ERR_UNSUPPORTED;
  }
}
