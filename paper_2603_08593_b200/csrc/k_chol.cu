// Blocked fp64 Cholesky solve of the normal equations (north_star subsystem (5)).
//
// One persistent cooperative kernel (k_chol_fused) runs the whole solve; the CTAs meet at a
// software grid barrier between phases, so the 2*N/32 phase boundaries cost ~1 us each instead of
// a kernel launch.  Right-looking blocked factorisation A = Lc Lc^T, block size NB = 32, on the
// augmented matrix [A b; b^T .]: carrying b as row N through the panel solves yields
// z = Lc^-1 b for free (the forward substitution), so only the back substitution Lc^T c = z remains.
//   phase 0       : copy the lower triangle of A and b into the workspace (inputs stay untouched)
//   panel phase k : every CTA factors the 32x32 diagonal block redundantly in shared memory
//                   (square-root-free elimination, scaled afterwards), then solves its rows of the
//                   panel X Lkk^T = A_ik, one row per warp, by substitution (backward stable; no
//                   explicit block inverse)
//   update phase k: trailing update A22 -= L21 L21^T on 32x32 tiles of the lower triangle
//   k_chol_back   : one 1024-thread CTA, blocked back substitution (a second, tiny launch)
// Square roots and divisions on the critical path are rsqrt + one fused Newton correction each
// (<= 1 ulp), which keeps the 32 dependent steps of a diagonal block short.
// info: 0, or the 1-based order of the first non-positive leading minor (no pivoting, no
// regularisation: DESIGN.md reading A9).
#include <mutex>
#include "sfft_common.cuh"

#define CH_NB 32
#define CH_THREADS 256
#define CH_WARPS (CH_THREADS / 32)

// Optional phase timestamps (development builds only: -DSFFT_CHOL_TIMING): CTA 0 records
// %globaltimer at every phase boundary into sfft_chol_dbg (k_chol_fused: entries 0.., its diagonal-block
// factorisation 200..204; k_chol_back: 100 + 3 per block).
#ifdef SFFT_CHOL_TIMING
__device__ unsigned long long sfft_chol_dbg[256];
#define CH_STAMP(i)                                                              \
  if (blockIdx.x == 0 && threadIdx.x == 0 && (i) < 256) {                        \
    unsigned long long t_;                                                       \
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_));                       \
    sfft_chol_dbg[i] = t_;                                                       \
  }
extern "C" int sfft_chol_dbg_read(unsigned long long* out, int n) {   // development builds only
  return (int)cudaMemcpyFromSymbol(out, sfft_chol_dbg, sizeof(unsigned long long) * (size_t)(n < 256 ? n : 256));
}
#else
#define CH_STAMP(i)
#endif

__device__ __forceinline__ double ld_cg(const double* p) { return __ldcg(p); }

// Grid barrier: monotonically increasing arrival counter; `target` is this CTA's private copy of
// the count that completes the next barrier.  Data written before the barrier is visible after it
// to loads that bypass L1 (ld_cg).
__device__ __forceinline__ void grid_barrier(unsigned* ctr, unsigned& target, unsigned nblocks) {
  __syncthreads();
  if (threadIdx.x == 0) {
    target += nblocks;
    __threadfence();
    atomicAdd(ctr, 1u);
    unsigned v;
    do {
      asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(ctr) : "memory");
    } while (v < target);
  }
  __syncthreads();
}

// sqrt and reciprocal-multiply with one fused correction step each
__device__ __forceinline__ void sqrt_and_rinv(double a, double& d, double& r) {
  r = rsqrt(a);
  d = a * r;
  d = fma(fma(-d, d, a), 0.5 * r, d);   // d = sqrt(a), < 1 ulp
  r = fma(fma(-d, r, 1.0), r, r);       // r = 1/d
}
__device__ __forceinline__ double div_by(double x, double d, double r) {  // x / d given r ~ 1/d
  const double q = x * r;
  return fma(fma(-q, d, x), r, q);
}

__device__ __forceinline__ double rcp_newton(double a) {  // 1/a for normal positive a, ~1 ulp
  // seed r0 (>= 20 bits), e = 1 - a r0; 1/a = r0 (1 + e + e^2 + O(e^3)): three dependent fp64 ops
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(a));
  const double e = fma(-a, r, 1.0);
  return fma(r, fma(e, e, e), r);
}

#define CH_PB 64              // panel width (two 32-blocks factored inside the CTA)
#define CH_LDS (CH_PB + 1)    // row pitch of the 64x64 shared arrays

// Cholesky of a 32x32 block (lower triangle, row pitch CH_LDS) in shared memory by the whole CTA.
// The 32 dependent steps run the square-root-free elimination a_ij -= a_ik a_jk / a_kk; the
// columns are scaled by 1/sqrt(pivot) afterwards, which gives exactly the Cholesky factor.
// Thread (warp w, lane j) keeps its elements (4w..4w+3, j) in registers for the whole elimination;
// per step only the pivot column travels through shared memory (double buffered, so one barrier
// per step).  srd receives 1/L_jj.  Returns the 0-based index of the first non-positive pivot (or
// -1); failed pivots are replaced by 1 so the work stays finite.
__device__ __forceinline__ int cta_potrf32(double* sd, double* srd, double (*colb)[CH_NB], int tid) {
  // TWO pivots per exchange step: columns k, k+1 travel through shared memory together and the
  // trailing elements are eliminated with the inverse of the 2x2 pivot block (one reciprocal of its
  // determinant on the dependent chain); column k+1 itself receives the single-pivot update, so the
  // stored values are exactly those of the column-by-column elimination.
  static_assert(CH_WARPS == 8, "row ownership below assumes 8 warps x 4 rows");
  const int j = tid & 31, i0 = (tid >> 5) * 4;
  double c[4];
  __syncthreads();  // sd was just filled by other threads
#pragma unroll
  for (int rr = 0; rr < 4; ++rr) c[rr] = sd[(i0 + rr) * CH_LDS + j];
  if (j < 2) {
#pragma unroll
    for (int rr = 0; rr < 4; ++rr) colb[j][i0 + rr] = c[rr];
  }
  int bad = -1;
#pragma unroll 1
  for (int k = 0; k < CH_NB; k += 2) {
    __syncthreads();
    const double* col0 = colb[(k & 2)];       // column k   (buffers 0,1 / 2,3 alternate)
    const double* col1 = colb[(k & 2) + 1];   // column k+1, not yet eliminated by column k
    double d00 = col0[k];
    const double d10 = col0[k + 1], d11 = col1[k + 1];
    const double aj0 = col0[j], aj1 = col1[j];
    const double2 p01 = *reinterpret_cast<const double2*>(col0 + i0);
    const double2 p23 = *reinterpret_cast<const double2*>(col0 + i0 + 2);
    const double2 q01 = *reinterpret_cast<const double2*>(col1 + i0);
    const double2 q23 = *reinterpret_cast<const double2*>(col1 + i0 + 2);
    if (!(d00 > 0.0)) {
      if (bad < 0) bad = k;
      d00 = 1.0;
    }
    double det = fma(d00, d11, -(d10 * d10));
    const double inv00 = rcp_newton(d00);
    if (!(det > 0.0)) {           // second pivot det/d00 not positive
      if (bad < 0) bad = k + 1;
      det = d00;
    }
    // numerators of D^-1 [aj0 aj1]^T, then the products with the thread's rows: all ahead of the
    // reciprocal of det
    const double n0 = fma(d11, aj0, -(d10 * aj1)), n1 = fma(d00, aj1, -(d10 * aj0));
    const double t0 = fma(p01.x, n0, q01.x * n1), t1 = fma(p01.y, n0, q01.y * n1);
    const double t2 = fma(p23.x, n0, q23.x * n1), t3 = fma(p23.y, n0, q23.y * n1);
    const double f = (j > k + 1) ? rcp_newton(det) : 0.0;   // columns <= k+1 take no 2x2 update
    c[0] = fma(-t0, f, c[0]);
    c[1] = fma(-t1, f, c[1]);
    c[2] = fma(-t2, f, c[2]);
    c[3] = fma(-t3, f, c[3]);
    if (j == k + 1) {             // column k+1: eliminated by column k alone
      const double g = d10 * inv00;
      c[0] = fma(-p01.x, g, c[0]);
      c[1] = fma(-p01.y, g, c[1]);
      c[2] = fma(-p23.x, g, c[2]);
      c[3] = fma(-p23.y, g, c[3]);
    }
    if ((j == k + 2 || j == k + 3) && k + 2 < CH_NB) {
      double* nxt = colb[((k + 2) & 2) + (j - k - 2)];
      *reinterpret_cast<double2*>(nxt + i0) = make_double2(c[0], c[1]);
      *reinterpret_cast<double2*>(nxt + i0 + 2) = make_double2(c[2], c[3]);
    }
  }
  // pivots (the diagonal as it stood when its column was eliminated) -> srd, then scale
  __syncthreads();
#pragma unroll
  for (int rr = 0; rr < 4; ++rr)
    if (i0 + rr == j) srd[j] = c[rr];
  __syncthreads();
  double piv = srd[j];
  if (!(piv > 0.0)) piv = 1.0;
  double d, r;
  sqrt_and_rinv(piv, d, r);
#pragma unroll
  for (int rr = 0; rr < 4; ++rr) {
    const int i = i0 + rr;
    sd[i * CH_LDS + j] = (i == j) ? d : (i > j ? div_by(c[rr], d, r) : 0.0);
  }
  __syncthreads();
  if (i0 == 0) srd[j] = r;
  __syncthreads();
  return bad;
}

// Cholesky of the 64x64 block sd (row pitch CH_LDS) by the whole CTA as a 2x2 recursion on
// 32-blocks: potrf(A11); X = A21 L11^-T by row substitution (4 rows per warp, interleaved chains);
// A22 -= X X^T; potrf(A22).  ss receives the column-scaled factor ss[i][j] = L[i][j] / L[j][j] and
// srd the reciprocals 1/L_jj of all 64 columns.  Returns the first bad pivot (or -1).
__device__ __forceinline__ int cta_potrf64(double* sd, double* ss, double* srd, double (*colb)[CH_NB], int tid) {
  const int lane = tid & 31, wrp = tid >> 5;
  CH_STAMP(200)
  int bad = cta_potrf32(sd, srd, colb, tid);
  CH_STAMP(201)
  // ss11 (needed by the substitution below)
  for (int e = tid; e < CH_NB * CH_NB; e += CH_THREADS) {
    const int i = e >> 5, j = e & 31;
    ss[i * CH_LDS + j] = sd[i * CH_LDS + j] * srd[j];
  }
  __syncthreads();
  {  // rows 32 + 4 wrp .. +3: x_j = a_j / L_jj, a_m -= a_j ss[m][j]
    double x[4];
#pragma unroll
    for (int rr = 0; rr < 4; ++rr) x[rr] = sd[(CH_NB + 4 * wrp + rr) * CH_LDS + lane];
#pragma unroll
    for (int j = 0; j < CH_NB - 1; ++j) {
      const double sj = ss[lane * CH_LDS + j];
#pragma unroll
      for (int rr = 0; rr < 4; ++rr) {
        const double aj = __shfl_sync(0xffffffffu, x[rr], j);
        if (lane > j) x[rr] = fma(-aj, sj, x[rr]);
      }
    }
    const double d = sd[lane * CH_LDS + lane], r = srd[lane];
#pragma unroll
    for (int rr = 0; rr < 4; ++rr) sd[(CH_NB + 4 * wrp + rr) * CH_LDS + lane] = div_by(x[rr], d, r);
  }
  __syncthreads();
  CH_STAMP(202)
  {  // A22 -= L21 L21^T on the lower triangle (outputs (ty, ty+16) x (tx, tx+16))
    const int tx = tid & 15, ty = tid >> 4;
    double acc[4] = {0.0, 0.0, 0.0, 0.0};
    const double* ri0 = sd + (CH_NB + ty) * CH_LDS, *ri1 = sd + (CH_NB + ty + 16) * CH_LDS;
    const double* rj0 = sd + (CH_NB + tx) * CH_LDS, *rj1 = sd + (CH_NB + tx + 16) * CH_LDS;
#pragma unroll
    for (int m = 0; m < CH_NB; ++m) {
      const double a0 = ri0[m], a1 = ri1[m], b0 = rj0[m], b1 = rj1[m];
      acc[0] = fma(a0, b0, acc[0]);
      acc[1] = fma(a0, b1, acc[1]);
      acc[2] = fma(a1, b0, acc[2]);
      acc[3] = fma(a1, b1, acc[3]);
    }
    __syncthreads();
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      const int i = ty + 16 * (q >> 1), j = tx + 16 * (q & 1);
      if (j <= i) sd[(CH_NB + i) * CH_LDS + CH_NB + j] -= acc[q];
    }
  }
  CH_STAMP(203)
  const int bad2 = cta_potrf32(sd + CH_NB * CH_LDS + CH_NB, srd + CH_NB, colb, tid);
  CH_STAMP(204)
  if (bad < 0 && bad2 >= 0) bad = CH_NB + bad2;
  for (int e = tid; e < CH_PB * CH_PB; e += CH_THREADS) {
    const int i = e >> 6, j = e & 63;
    if (i >= CH_NB || j >= CH_NB) ss[i * CH_LDS + j] = (j <= i) ? sd[i * CH_LDS + j] * srd[j] : 0.0;
  }
  __syncthreads();
  return bad;
}

__global__ void __launch_bounds__(CH_THREADS, 1)
k_chol_fused(const double* __restrict__ A, const double* __restrict__ b, double* Lw,
             int N, int ld, int* info, unsigned* bar) {
  // shared memory: panel phase  sd[64][65] (factored diagonal block), ss[64][65] (column-scaled);
  //                update phase pi[32][65], pj[32][65] (aliasing sd / ss)
  extern __shared__ __align__(16) double ch_smem[];
  double* sd = ch_smem;
  double* ss = sd + CH_PB * CH_LDS;
  double* pi = sd;
  double* pj = ss;
  __shared__ double srd[CH_PB];                    // reciprocals of the diagonal
  __shared__ __align__(16) double colb[4][CH_NB];  // pivot column exchange of cta_potrf32 (2 x 2 columns)
  const int tid = threadIdx.x, lane = tid & 31, wrp = tid >> 5;
  const unsigned nblocks = gridDim.x;
  unsigned target = 0;

  // ---- phase 0: workspace <- lower triangle of A, row N <- b
  {
    const size_t total = (size_t)(N + 1) * N;
    if (blockIdx.x == 0 && tid == 0 && info) *info = 0;
    // eight elements per thread and round, all requested before the first store (one memory latency per round)
    const unsigned stride = nblocks * CH_THREADS;
    for (unsigned e0 = blockIdx.x * CH_THREADS + tid; e0 < (unsigned)total; e0 += 8u * stride) {
      double val[8];
      int dst[8];
#pragma unroll
      for (int q = 0; q < 8; ++q) {
        const unsigned e = e0 + (unsigned)q * stride;
        dst[q] = -1;
        val[q] = 0.0;
        if (e < (unsigned)total) {
          const int i = (int)(e / (unsigned)N), j = (int)(e - (unsigned)i * (unsigned)N);
          if (i == N) { dst[q] = N * ld + j; val[q] = b[j]; }
          else if (j <= i) { dst[q] = i * ld + j; val[q] = A[e]; }
        }
      }
#pragma unroll
      for (int q = 0; q < 8; ++q)
        if (dst[q] >= 0) Lw[dst[q]] = val[q];
    }
  }
  CH_STAMP(0)
  grid_barrier(bar, target, nblocks);
  CH_STAMP(1)
  int stamp = 2;
  (void)stamp;

  const int gw = blockIdx.x * CH_WARPS + wrp, ngw = nblocks * CH_WARPS;
  for (int k0 = 0; k0 < N; k0 += CH_PB) {
    const int nb = min(CH_PB, N - k0);
    const int rbelow = k0 + nb;                 // first row below the diagonal block
    // ---- panel phase: CTAs that own panel rows (and CTA 0) factor the diagonal block
    const bool has_rows = blockIdx.x * CH_WARPS < (N + 1 - rbelow);
    // the factored block is written back (after the grid barrier) by a CTA that owns no panel rows when
    // there is one, else by CTA 0
    const unsigned storer = (nblocks - 1) * CH_WARPS >= (unsigned)(N + 1 - rbelow) ? nblocks - 1 : 0u;
    if (has_rows || blockIdx.x == storer) {
      // the warp's first panel row is final already: request it now, its L2 latency hides under the factor
      const int row0 = rbelow + gw;
      double pre0 = 0.0, pre1 = 0.0;
      if (row0 <= N) {
        const double* src = Lw + (size_t)row0 * ld + k0;
        if (lane < nb) pre0 = ld_cg(src + lane);
        if (lane + CH_NB < nb) pre1 = ld_cg(src + lane + CH_NB);
      }
      {
        // all of the thread's 16 elements are requested before the first one is stored: one L2 latency
        double blk[CH_PB * CH_PB / CH_THREADS];
#pragma unroll
        for (int q = 0; q < CH_PB * CH_PB / CH_THREADS; ++q) {
          const int e = tid + q * CH_THREADS, i = e >> 6, j = e & 63;
          blk[q] = (i < nb && j <= i) ? ld_cg(Lw + (size_t)(k0 + i) * ld + k0 + j) : (i == j ? 1.0 : 0.0);
        }
#pragma unroll
        for (int q = 0; q < CH_PB * CH_PB / CH_THREADS; ++q) {
          const int e = tid + q * CH_THREADS, i = e >> 6, j = e & 63;
          sd[i * CH_LDS + j] = blk[q];
        }
      }
      const int bad = cta_potrf64(sd, ss, srd, colb, tid);
      if (bad >= 0 && bad < nb && blockIdx.x == storer && tid == 0 && info) atomicCAS(info, 0, k0 + bad + 1);
      CH_STAMP(stamp + 0)
      // rows below (including the rhs row N): one row per warp, lane holds entries lane and lane+32.
      // x_j = a_j / L_jj, a_m -= x_j L_mj = a_j ss[m][j]: per step one shuffle and one fma on the
      // dependent chain; the divisions are off it
      for (int row = rbelow + gw; row <= N; row += ngw) {
        double* src = Lw + (size_t)row * ld + k0;
        double x0 = pre0, x1 = pre1;
        if (row != row0) {
          x0 = (lane < nb) ? ld_cg(src + lane) : 0.0;
          x1 = (lane + CH_NB < nb) ? ld_cg(src + lane + CH_NB) : 0.0;
        }
        const double* s0 = ss + lane * CH_LDS, *s1 = ss + (lane + CH_NB) * CH_LDS;
#pragma unroll
        for (int j = 0; j < CH_NB; ++j) {
          const double aj = __shfl_sync(0xffffffffu, x0, j);
          if (lane > j) x0 = fma(-aj, s0[j], x0);
          x1 = fma(-aj, s1[j], x1);
        }
#pragma unroll
        for (int j = 0; j < CH_NB - 1; ++j) {
          const double aj = __shfl_sync(0xffffffffu, x1, j);
          if (lane > j) x1 = fma(-aj, s1[CH_NB + j], x1);
        }
        if (lane < nb) src[lane] = div_by(x0, sd[lane * CH_LDS + lane], srd[lane]);
        if (lane + CH_NB < nb)
          src[lane + CH_NB] = div_by(x1, sd[(lane + CH_NB) * CH_LDS + lane + CH_NB], srd[lane + CH_NB]);
      }
    }
    CH_STAMP(stamp + 1)
    grid_barrier(bar, target, nblocks);
    CH_STAMP(stamp + 2)
    // The factored diagonal block is written back only now: before the barrier the other CTAs were still
    // reading the UNFACTORED block from the same addresses.  The storer's copy in shared memory is intact
    // until the update phase below reuses the buffers; nothing in this kernel reads the block again
    // (k_chol_back does), so the store is off every critical path.
    if (blockIdx.x == storer) {
      for (int e = tid; e < CH_PB * CH_PB; e += CH_THREADS) {
        const int i = e >> 6, j = e & 63;
        if (i < nb && j <= i) Lw[(size_t)(k0 + i) * ld + k0 + j] = sd[i * CH_LDS + j];
      }
      __syncthreads();
    }
    // ---- update phase: 32x32 tiles (ti, tj), tj <= ti, of the trailing matrix starting at r0,
    //      A22 -= L21 L21^T with the panel's 64 columns
    const int r0 = k0 + CH_PB;
    if (r0 <= N) {
      const int T = (N + 1 - r0 + CH_NB - 1) / CH_NB;
      const int ntile = T * (T + 1) / 2;
      const int tx = tid & 15, ty = tid >> 4;      // outputs (ty, ty+16) x (tx, tx+16)
      double gpi[8], gpj[8], cur[4];
      int ti = 0, tj = 0;
      auto decode = [&](int t, int& oi, int& oj) {   // t -> (ti, tj): ti(ti+1)/2 <= t
        int q = (int)((sqrt(8.0 * t + 1.0) - 1.0) * 0.5);
        while ((q + 1) * (q + 2) / 2 <= t) ++q;
        while (q * (q + 1) / 2 > t) --q;
        oi = q; oj = t - q * (q + 1) / 2;
      };
      auto fetch = [&](int fi, int fj) {
#pragma unroll
        for (int q = 0; q < 8; ++q) {
          const int e = tid + q * CH_THREADS, r = e >> 6, m = e & 63;
          const int gi = r0 + fi * CH_NB + r, gj = r0 + fj * CH_NB + r;
          gpi[q] = (gi <= N) ? ld_cg(Lw + (size_t)gi * ld + k0 + m) : 0.0;
          gpj[q] = (gj < N) ? ld_cg(Lw + (size_t)gj * ld + k0 + m) : 0.0;
        }
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          const int gi = r0 + fi * CH_NB + ty + 16 * (q >> 1), gj = r0 + fj * CH_NB + tx + 16 * (q & 1);
          cur[q] = (gi <= N && gj < N && gj <= gi) ? ld_cg(Lw + (size_t)gi * ld + gj) : 0.0;
        }
      };
      int t = blockIdx.x;
      if (t < ntile) { decode(t, ti, tj); fetch(ti, tj); }
      while (t < ntile) {
        __syncthreads();
#pragma unroll
        for (int q = 0; q < 8; ++q) {
          const int e = tid + q * CH_THREADS, r = e >> 6, m = e & 63;
          pi[r * CH_LDS + m] = gpi[q];
          pj[r * CH_LDS + m] = gpj[q];
        }
        double c0[4] = {cur[0], cur[1], cur[2], cur[3]};
        const int ci = ti, cj = tj;
        __syncthreads();
        t += nblocks;
        if (t < ntile) { decode(t, ti, tj); fetch(ti, tj); }
        double acc[4] = {0.0, 0.0, 0.0, 0.0};
        const double* a0p = pi + ty * CH_LDS, *a1p = pi + (ty + 16) * CH_LDS;
        const double* b0p = pj + tx * CH_LDS, *b1p = pj + (tx + 16) * CH_LDS;
#pragma unroll
        for (int m = 0; m < CH_PB; ++m) {
          const double a0 = a0p[m], a1 = a1p[m], b0 = b0p[m], b1 = b1p[m];
          acc[0] = fma(a0, b0, acc[0]);
          acc[1] = fma(a0, b1, acc[1]);
          acc[2] = fma(a1, b0, acc[2]);
          acc[3] = fma(a1, b1, acc[3]);
        }
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          const int gi = r0 + ci * CH_NB + ty + 16 * (q >> 1), gj = r0 + cj * CH_NB + tx + 16 * (q & 1);
          if (gi <= N && gj < N && gj <= gi) Lw[(size_t)gi * ld + gj] = c0[q] - acc[q];
        }
      }
      CH_STAMP(stamp + 3)
      grid_barrier(bar, target, nblocks);
      CH_STAMP(stamp + 4)
    }
    stamp += 5;
  }

  // last CTA out resets the barrier counter for the next launch
  __syncthreads();
  if (tid == 0) {
    unsigned* done = bar + 1;
    const unsigned old = atomicInc(done, nblocks - 1);
    if (old == nblocks - 1) { __threadfence(); *bar = 0u; }
  }
}

// Back substitution Lc^T c = z; z is row N of the workspace.  Per 64-block (last to first): the block's
// triangular system is solved by warp 0 (lane m holds r_m and r_{m+32}; row-scaled factor, so one shuffle
// and one or two fmas per dependent step), then every thread j < k0 updates
// r_j -= sum_i L[k0+i][j] x_i in two batches of 32 loads issued together (coalesced along j).  64-wide
// blocks halve the number of (barrier, L2 round trip) pairs of the 32-wide version (80 -> 45 us at N = 732).
#define CHB_NB 64
#define CHB_TH 512   // 128 registers per thread: the 32 entries of a batch stay in registers
__global__ void __launch_bounds__(CHB_TH, 1) k_chol_back(const double* __restrict__ Lw, double* c, int N, int ld) {
  extern __shared__ double sm[];
  double* r = sm;                             // N running right-hand side
  double* ls = sm + N;                        // 64 x 65 diagonal factor
  double* rd = ls + CHB_NB * (CHB_NB + 1);    // reciprocals of its diagonal
  double* cb = rd + CHB_NB;                   // 64 solved values of the current block
  const int tid = threadIdx.x, lane = tid & 31;
  for (int j = tid; j < N; j += CHB_TH) r[j] = Lw[(size_t)N * ld + j];
  const int nblk = (N + CHB_NB - 1) / CHB_NB;
  {
    const int k0 = (nblk - 1) * CHB_NB, nb = N - k0;
    constexpr int NQ0 = CHB_NB * CHB_NB / CHB_TH;
    double blk[NQ0];   // all requested before the first store: one L2 latency
#pragma unroll
    for (int q = 0; q < NQ0; ++q) {
      const int e = tid + q * CHB_TH, i = e >> 6, j = e & 63;
      blk[q] = (i < nb && j <= i) ? Lw[(size_t)(k0 + i) * ld + k0 + j] : (i == j ? 1.0 : 0.0);
    }
#pragma unroll
    for (int q = 0; q < NQ0; ++q) {
      const int e = tid + q * CHB_TH;
      ls[(e >> 6) * (CHB_NB + 1) + (e & 63)] = blk[q];
    }
  }
  __syncthreads();
  CH_STAMP(100)
  for (int kb = nblk - 1; kb >= 0; --kb) {
    const int k0 = kb * CHB_NB;
    const int nb = min(CHB_NB, N - k0);
    if (tid < 32) {
      // x_j = r_j / L_jj, r_m -= L[j][m] x_j = r_j (L[j][m] / L[j][j]): the scalings and the final divisions are
      // off the dependent chain
      const double d0 = ls[lane * (CHB_NB + 1) + lane], d1 = ls[(lane + 32) * (CHB_NB + 1) + lane + 32];
      const double r0 = 1.0 / d0, r1 = 1.0 / d1;
      rd[lane] = r0; rd[lane + 32] = r1;
      __syncwarp();
      double rm0 = (lane < nb) ? r[k0 + lane] : 0.0, rm1 = (lane + 32 < nb) ? r[k0 + lane + 32] : 0.0;
#pragma unroll
      for (int j = CHB_NB - 1; j >= 32; --j) {
        const double rdj = rd[j];
        const double s0 = ls[j * (CHB_NB + 1) + lane] * rdj, s1 = ls[j * (CHB_NB + 1) + lane + 32] * rdj;
        const double rj = __shfl_sync(0xffffffffu, rm1, j - 32);
        if (lane + 32 < j) rm1 = fma(-s1, rj, rm1);
        rm0 = fma(-s0, rj, rm0);
      }
#pragma unroll
      for (int j = 31; j >= 0; --j) {
        const double s0 = ls[j * (CHB_NB + 1) + lane] * rd[j];
        const double rj = __shfl_sync(0xffffffffu, rm0, j);
        if (lane < j) rm0 = fma(-s0, rj, rm0);
      }
      rm0 = div_by(rm0, d0, r0);
      rm1 = div_by(rm1, d1, r1);
      cb[lane] = (lane < nb) ? rm0 : 0.0;
      cb[lane + 32] = (lane + 32 < nb) ? rm1 : 0.0;
      if (lane < nb) c[k0 + lane] = rm0;
      if (lane + 32 < nb) c[k0 + lane + 32] = rm1;
    }
    CH_STAMP(101 + 3 * kb)
    // the next diagonal block is requested while warp 0 solves
    constexpr int NQ = CHB_NB * CHB_NB / CHB_TH;
    double nxt[NQ];
#pragma unroll
    for (int q = 0; q < NQ; ++q) nxt[q] = 0.0;
    if (kb > 0) {
#pragma unroll
      for (int q = 0; q < NQ; ++q) {
        const int e = tid + q * CHB_TH, i = e >> 6, j = e & 63;
        nxt[q] = (j <= i) ? __ldcg(Lw + (size_t)(k0 - CHB_NB + i) * ld + k0 - CHB_NB + j) : 0.0;
      }
    }
    __syncthreads();
    if (kb > 0) {
#pragma unroll
      for (int q = 0; q < NQ; ++q) {
        const int e = tid + q * CHB_TH;
        ls[(e >> 6) * (CHB_NB + 1) + (e & 63)] = nxt[q];
      }
    }
    CH_STAMP(102 + 3 * kb)
    for (int j = tid; j < k0; j += CHB_TH) {
      double a0 = r[j], a1 = 0.0;
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        double v[32];
#pragma unroll
        for (int i = 0; i < 32; ++i) v[i] = (32 * h + i < nb) ? __ldcg(Lw + (size_t)(k0 + 32 * h + i) * ld + j) : 0.0;
#pragma unroll
        for (int i = 0; i < 32; i += 2) {
          a0 = fma(-v[i], cb[32 * h + i], a0);
          a1 = fma(-v[i + 1], cb[32 * h + i + 1], a1);
        }
      }
      r[j] = a0 + a1;
    }
    __syncthreads();
    CH_STAMP(103 + 3 * kb)
  }
}

sfft_status sfft_launch_solve(sfft_plan* p, const double* A, const double* b, double* c, int* info,
                              cudaStream_t st, int* nl) {
  int N = p->N, ld = p->ldL;
  double* Lw = p->Lw;
  unsigned* bar = p->cholBar;
  void* args[] = {(void*)&A, (void*)&b, (void*)&Lw, (void*)&N, (void*)&ld, (void*)&info, (void*)&bar};
  // every CTA must be resident for the grid barrier: cooperative launch, one CTA per SM at most
  int grid = p->num_sms;
  const int rows = N + 1, maxUseful = (rows + CH_WARPS - 1) / CH_WARPS;
  const int T = (N + CH_NB - 1) / CH_NB, tiles = T * (T + 1) / 2;
  int want = maxUseful > tiles ? maxUseful : tiles;
  if (want < 1) want = 1;
  if (grid > want) grid = want;
  if (p->cholMaxCtas > 0 && grid > p->cholMaxCtas) grid = p->cholMaxCtas;
  // a prepared subtract stage is running on the side stream: leave about a third of the SMs to it
  // (the solve is latency-bound: 96 instead of 148 CTAs cost it ~2 %)
  if (p->cholMaxCtas == 0 && p->prepValid && grid > (p->num_sms * 13) / 20) grid = (p->num_sms * 13) / 20;
  const size_t smemF = (size_t)2 * CH_PB * CH_LDS * sizeof(double);
  SFFT_CUDA_TRY(cudaFuncSetAttribute(k_chol_fused, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smemF));
  SFFT_CUDA_TRY(cudaLaunchCooperativeKernel((const void*)k_chol_fused, dim3(grid), dim3(CH_THREADS), args, smemF, st));
  ++*nl;
  const size_t smem = ((size_t)N + CHB_NB * (CHB_NB + 1) + 2 * CHB_NB) * sizeof(double);
  SFFT_CUDA_TRY(cudaFuncSetAttribute(k_chol_back, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  k_chol_back<<<1, CHB_TH, smem, st>>>(Lw, c, N, ld);
  SFFT_LAUNCH_CHECK();
  ++*nl;
  return SFFT_OK;
}

// ------------------------------------------------------------------------------------------------
// sfft_solve_static (include/sfft.h): the same two kernels with the factorisation workspace in a static
// device array, for callers that must not allocate.  Layout of the array: (N + 1) rows of pitch ld =
// round-up(N + 1, 4) doubles (the layout sfft_launch_solve uses in a plan's Lw), then, at a fixed offset
// past the largest workspace, the two grid-barrier words of k_chol_fused.
#define NA_MAXN SFFT_SOLVE_STATIC_MAX_N
#define NA_LD ((NA_MAXN + 1 + 3) & ~3)
#define NA_WORK ((size_t)(NA_MAXN + 1) * NA_LD)      // doubles
#define NA_TOTAL (NA_WORK + 32)                      // + 256 bytes for the barrier words
static __device__ __align__(256) double sfft_static_scratch[NA_TOTAL];

#define NA_MAXDEV 64
namespace {
struct NaDevice {
  double* scratch;   // device address of sfft_static_scratch on this device
  int sms;
  bool ready;
};
NaDevice na_dev[NA_MAXDEV];   // zero-initialised
std::mutex na_mutex;
}  // namespace

extern "C" sfft_status sfft_solve_static(const double* A, const double* b, int N, double* coeffs, int* info,
                                         void* stream) {
  if (!A || !b || !coeffs || N < 1) return SFFT_ERR_INVALID_ARG;
  if (N > NA_MAXN) return SFFT_ERR_UNSUPPORTED;
  if (cudaPeekAtLastError() != cudaSuccess) return SFFT_ERR_CUDA;
  cudaStream_t st = (cudaStream_t)stream;
  int dev = -1;
  SFFT_CUDA_TRY(cudaGetDevice(&dev));
  if (dev < 0 || dev >= NA_MAXDEV) return SFFT_ERR_UNSUPPORTED;
  NaDevice& nd = na_dev[dev];
  std::lock_guard<std::mutex> lock(na_mutex);   // set-up once per device; the launches below stay ordered per caller
  if (!nd.ready) {
    // once per device, with that device current: in host code the array's name is only a handle, the
    // device address comes from the runtime
    double* ptr = nullptr;
    int sms = 0;
    SFFT_CUDA_TRY(cudaGetSymbolAddress((void**)&ptr, sfft_static_scratch));
    SFFT_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    if (!ptr || sms < 1) return SFFT_ERR_CUDA;
    nd.scratch = ptr;
    nd.sms = sms;
    nd.ready = true;
  }
  double* Lw = nd.scratch;
  unsigned* bar = reinterpret_cast<unsigned*>(nd.scratch + NA_WORK);
  int ld = (N + 1 + 3) & ~3;
  // the barrier words must start at zero whatever an earlier (possibly aborted) call left there
  SFFT_CUDA_TRY(cudaMemsetAsync(bar, 0, 2 * sizeof(unsigned), st));
  void* args[] = {(void*)&A, (void*)&b, (void*)&Lw, (void*)&N, (void*)&ld, (void*)&info, (void*)&bar};
  int grid = nd.sms;   // cooperative launch: one CTA per SM at most
  const int rows = N + 1, maxUseful = (rows + CH_WARPS - 1) / CH_WARPS;
  const int T = (N + CH_NB - 1) / CH_NB, tiles = T * (T + 1) / 2;
  int want = maxUseful > tiles ? maxUseful : tiles;
  if (want < 1) want = 1;
  if (grid > want) grid = want;
  const size_t smemF = (size_t)2 * CH_PB * CH_LDS * sizeof(double);
  SFFT_CUDA_TRY(cudaFuncSetAttribute(k_chol_fused, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smemF));
  SFFT_CUDA_TRY(cudaLaunchCooperativeKernel((const void*)k_chol_fused, dim3(grid), dim3(CH_THREADS), args, smemF, st));
  const size_t smem = ((size_t)N + CHB_NB * (CHB_NB + 1) + 2 * CHB_NB) * sizeof(double);
  SFFT_CUDA_TRY(cudaFuncSetAttribute(k_chol_back, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  k_chol_back<<<1, CHB_TH, smem, st>>>(Lw, coeffs, N, ld);
  SFFT_LAUNCH_CHECK();
  return SFFT_OK;
}
