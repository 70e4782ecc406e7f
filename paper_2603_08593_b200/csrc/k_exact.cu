// Exact unmasked-pixel objective (BASELINE.json north_star: "the coefficients
// minimise sum D^2 over unmasked pixels").  With g(x) the row of the design matrix of the UNMASKED
// images at pixel x,
//     A_ex = sum_{x unmasked} g g^T = A(mask = NULL) - sum_{x masked} g(x) g(x)^T,
//     b_ex = b(mask = NULL) - sum_{x masked} g(x) S(x).
// sfft_build_system_exact runs the ordinary (Fourier) build with no mask and then subtracts the
// masked pixels' rank-one terms: a symmetric rank-K update (K = number of masked pixels, 74 k at the
// full CCD) of the N x N matrix, C = Gm^T Gm with the S values riding as column N.
//
//  k_mk_rows / k_mk_scan : ordered list of the masked pixels (per-row counts, scan, fill).
//  k_exact_syrk          : cooperative kernel, one CTA = one 128 x 128 tile of the lower triangle x
//                          one slice of the pixel list.  Per chunk of 16384 masked pixels all CTAs
//                          first generate the chunk's rows of Gm once (coalesced), then each adds its
//                          slice to its tile with the fp64 tensor path (mma.sync m8n8k4, warp tiles of
//                          64 x 32: a dense contraction is where tensor cores belong), double-buffered
//                          16 x 128 panels, the next panels' loads in flight under the current one's MMAs.
//  k_exact_apply         : adds the slices in order and subtracts the tile from A (both triangles), b.
// Every sum has a fixed order, so the result is reproducible run to run.
#include "sfft_common.cuh"

#define EX_T 128      // tile edge
#define EX_KS 16      // pixels per panel
#define EX_TH 256
#define EX_PITCH (EX_T + 4)   // panel row pitch in doubles: the (row, k) lanes of an mma fragment hit distinct banks
#define EX_KC 16384  // masked pixels per chunk of the generated rows
#ifndef EX_UNR
#define EX_UNR 4
#endif
constexpr int EXU = EX_UNR;   // unroll factor of the panel loop

// ---- masked-pixel list ---------------------------------------------------------------------------
template <bool FILL>
__global__ void __launch_bounds__(256) k_mk_rows(const unsigned char* __restrict__ mask, int H, int W, int* cnt,
                                                 const int* __restrict__ off, int* list) {
  const int lane = threadIdx.x & 31;
  const int y = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (y >= H) return;
  const int base = FILL ? off[y] : 0;
  int total = 0;
  for (int k = 0; k < (W + 511) / 512; ++k) {   // uniform trip count for the shuffles
    const int x0 = k * 512 + lane * 16;
    unsigned mk = 0u;
    if (x0 < W) {   // W is a multiple of 32
      const uint4 m16 = *reinterpret_cast<const uint4*>(mask + (size_t)y * W + x0);
      const unsigned wd[4] = {m16.x, m16.y, m16.z, m16.w};
#pragma unroll
      for (int q = 0; q < 4; ++q)
#pragma unroll
        for (int i = 0; i < 4; ++i)
          if ((wd[q] >> (8 * i)) & 0xffu) mk |= 1u << (4 * q + i);
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

__global__ void __launch_bounds__(1024) k_mk_scan(const int* __restrict__ cnt, int* off, int H) {
  __shared__ int part[1024];
  const int tid = threadIdx.x;
  const int per = (H + 1023) / 1024;
  int loc[4] = {0, 0, 0, 0}, sum = 0;
  for (int i = 0; i < per; ++i) {
    const int y = tid * per + i;
    loc[i] = y < H ? cnt[y] : 0;
    sum += loc[i];
  }
  part[tid] = sum;
  __syncthreads();
  for (int o = 1; o < 1024; o <<= 1) {
    const int t = tid >= o ? part[tid - o] : 0;
    __syncthreads();
    part[tid] += t;
    __syncthreads();
  }
  int run = part[tid] - sum;
  for (int i = 0; i < per; ++i) {
    const int y = tid * per + i;
    if (y < H) off[y] = run;
    run += loc[i];
  }
  if (tid == 1023) off[H] = part[1023];
}

// ---- symmetric rank-K update from the masked pixels -----------------------------------------------
struct ExactParams {
  const double* R;
  const double* S;
  const int* list;    // masked pixels y*W + x, ascending
  const int* off;     // off[H] = their number
  double* Cpart;      // [KSplit][ntiles][EX_T*EX_T]
  double* Gm;         // [EX_KC][Npad] rows of the design matrix of the current chunk of masked pixels
  unsigned* bar;      // grid-barrier counters (arrivals, finished CTAs)
  int H, W, w, L, TK, TB, N, ntb, KSplit, log2W;
  int monoK[SFFT_MAX_T][2], monoB[SFFT_MAX_T][2];
};

// column n of the design matrix: 0 = padding, 1 = kernel column (p, q, u, v), 2 = background (p, q),
// 3 = the S values (column N)
struct ExCol { int kind, p, q, u, v; };
__device__ __forceinline__ ExCol ex_column(const ExactParams& P, int n) {
  ExCol c = {0, 0, 0, 0, 0};
  const int nK = P.L * P.TK, S1 = 2 * P.w + 1;
  if (n < nK) {
    const int t = n / P.L, s = n - t * P.L;
    c.kind = 1; c.p = P.monoK[t][0]; c.q = P.monoK[t][1]; c.u = s % S1 - P.w; c.v = s / S1 - P.w;
  } else if (n < P.N) {
    c.kind = 2; c.p = P.monoB[n - nK][0]; c.q = P.monoB[n - nK][1];
  } else if (n == P.N) {
    c.kind = 3;
  }
  return c;
}

// software grid barrier (cooperative launch: every CTA is resident); data written before it is
// visible after it to loads that bypass L1
__device__ __forceinline__ void ex_grid_barrier(unsigned* ctr, unsigned& target, unsigned nblocks) {
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

// element (pixel, column n) of the masked rows of the design matrix
__device__ __forceinline__ double ex_element(const ExactParams& P, int pixel, int n) {
  const ExCol col = ex_column(P, n);
  if (col.kind == 0) return 0.0;
  const int W = P.W, H = P.H;
  const int y = pixel >> P.log2W, x = pixel & (W - 1);   // W is a power of two
  if (col.kind == 3) return P.S[(size_t)y * W + x];
  const int xs = (x - col.u + W) & (W - 1), ys = (y - col.v + H) & (H - 1);   // u = v = 0 for background columns
  const double pw = ipow((double)(2 * xs + 1 - W) / (double)W, col.p) * ipow((double)(2 * ys + 1 - H) / (double)H, col.q);
  return col.kind == 1 ? pw * P.R[(size_t)ys * W + xs] : pw;
}

// Cooperative kernel, grid = (tiles of the lower triangle) x (slices).  The pixel list is walked in
// chunks of EX_KC pixels: all CTAs first write the chunk's rows Gm[k][Npad] (every element generated
// once, coalesced along the columns), meet at a grid barrier, then every CTA adds its slice of the
// chunk to its 128 x 128 tile (mma.sync m8n8k4 on 64 x 32 warp tiles; the next 16-row panels travel
// global -> registers under the current panel's MMAs, then into the other shared buffer), and a
// second barrier frees the chunk buffer.
__global__ void __launch_bounds__(EX_TH, 1) k_exact_syrk(ExactParams P) {
  extern __shared__ __align__(16) double ex_pan[];   // [2 buffers][2 blocks][EX_KS][EX_T]
  const int tid = threadIdx.x;
  const unsigned nblocks = gridDim.x * gridDim.y;
  unsigned target = 0;
  int ti = 0;
  {
    const int t = blockIdx.x;
    while ((ti + 1) * (ti + 2) / 2 <= t) ++ti;
  }
  const int tj = blockIdx.x - ti * (ti + 1) / 2;
  const int nm = P.off[P.H];
  if (nm == 0) return;        // empty list (uniform over the grid): nothing is written, k_exact_apply skips it too
  const int Npad = P.ntb * EX_T;
  // product role: 8 warps as 2 (rows) x 4 (columns), warp tile 64 x 32 = 8 x 4 mma tiles of
  // m8n8k4 (fp64 tensor path, mma.sync): lane holds A[row = lane/4][k = lane%4], B[k = lane%4][col = lane/4]
  // and C[row = lane/4][2 (lane%4), +1] of every tile -- one shared load feeds 8 multiply-adds per
  // thread instead of 4 in the scalar form, which was bound by the shared-memory pipe
  const int lane = tid & 31, wrp = tid >> 5;
  const int wr = (wrp >> 2) * 64, wc = (wrp & 3) * 32;
  const int fr = lane >> 2, fk = lane & 3;
  double acc[8][4][2];
#pragma unroll
  for (int mt = 0; mt < 8; ++mt)
#pragma unroll
    for (int nt = 0; nt < 4; ++nt) acc[mt][nt][0] = acc[mt][nt][1] = 0.0;

  for (int c0 = 0; c0 < nm; c0 += EX_KC) {
    const int kc = min(EX_KC, nm - c0);
    // ---- phase G: the chunk's rows of the design matrix
    {
      const size_t total = (size_t)kc * Npad;
      const size_t gtid = ((size_t)blockIdx.y * gridDim.x + blockIdx.x) * EX_TH + tid;
      for (size_t e = gtid; e < total; e += (size_t)nblocks * EX_TH) {
        const int k = (int)(e / Npad), n = (int)(e - (size_t)k * Npad);
        P.Gm[e] = ex_element(P, P.list[c0 + k], n);
      }
    }
    ex_grid_barrier(P.bar, target, nblocks);
    // ---- phase S: this CTA's slice [kbeg, kend) of the chunk
    const int slice = (((kc + P.KSplit - 1) / P.KSplit) + EX_KS - 1) / EX_KS * EX_KS;
    const int kbeg = blockIdx.y * slice, kend = min(kc, kbeg + slice);
    // staging: 2 blocks x 16 rows x 128 columns = 2048 double2 per panel pair, 8 per thread
    double2 stg[8];
    auto fetch = [&](int k0) {
#pragma unroll
      for (int q = 0; q < 8; ++q) {
        const int e = tid + q * EX_TH;                 // 0..2047
        const int blk = e >> 10, r = (e >> 6) & 15, c2 = e & 63;
        const int k = k0 + r;
        stg[q] = k < kend ? __ldcg(reinterpret_cast<const double2*>(P.Gm + (size_t)k * Npad + (blk == 0 ? ti : tj) * EX_T) + c2)
                          : make_double2(0.0, 0.0);
      }
    };
    auto stash = [&](int buf) {
#pragma unroll
      for (int q = 0; q < 8; ++q) {
        const int e = tid + q * EX_TH;
        const int blk = e >> 10, r = (e >> 6) & 15, c2 = e & 63;
        reinterpret_cast<double2*>(ex_pan + ((size_t)(buf * 2 + blk) * EX_KS + r) * EX_PITCH)[c2] = stg[q];
      }
    };
    if (kbeg < kend) {
      fetch(kbeg);
      stash(0);
    }
    __syncthreads();
    int buf = 0;
    for (int k0 = kbeg; k0 < kend; k0 += EX_KS, buf ^= 1) {
      const bool more = k0 + EX_KS < kend;
      if (more) fetch(k0 + EX_KS);
      const double* pa = ex_pan + ((size_t)(buf * 2 + 0) * EX_KS + fk) * EX_PITCH + wr + fr;
      const double* pb = ex_pan + ((size_t)(buf * 2 + 1) * EX_KS + fk) * EX_PITCH + wc + fr;
#pragma unroll
      for (int k4 = 0; k4 < EX_KS; k4 += 4) {
        double a[8], b[4];
#pragma unroll
        for (int mt = 0; mt < 8; ++mt) a[mt] = pa[k4 * EX_PITCH + 8 * mt];
#pragma unroll
        for (int nt = 0; nt < 4; ++nt) b[nt] = pb[k4 * EX_PITCH + 8 * nt];
#pragma unroll
        for (int mt = 0; mt < 8; ++mt)
#pragma unroll
          for (int nt = 0; nt < 4; ++nt)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                         : "+d"(acc[mt][nt][0]), "+d"(acc[mt][nt][1])
                         : "d"(a[mt]), "d"(b[nt]));
      }
      if (more) stash(buf ^ 1);
      __syncthreads();
    }
    if (c0 + EX_KC < nm) ex_grid_barrier(P.bar, target, nblocks);   // the chunk buffer is rewritten next
  }
  double* out = P.Cpart + ((size_t)blockIdx.y * gridDim.x + blockIdx.x) * EX_T * EX_T;
#pragma unroll
  for (int mt = 0; mt < 8; ++mt)
#pragma unroll
    for (int nt = 0; nt < 4; ++nt)
      *reinterpret_cast<double2*>(out + (size_t)(wr + 8 * mt + fr) * EX_T + wc + 8 * nt + 2 * fk) =
          make_double2(acc[mt][nt][0], acc[mt][nt][1]);
  // last CTA out resets the barrier counter for the next launch
  __syncthreads();
  if (tid == 0) {
    unsigned* done = P.bar + 1;
    const unsigned old = atomicInc(done, nblocks - 1);
    if (old == nblocks - 1) { __threadfence(); *P.bar = 0u; }
  }
}

// A[i][j] += sign * sum_ks C[i][j] (both triangles from the same sum), b[i] += sign * sum_ks C[N][i]; sign = -1 or +1
__global__ void __launch_bounds__(256) k_exact_apply(const double* __restrict__ Cpart, double* A, double* b, int N,
                                                     int ntiles, int KSplit, double sign, const int* __restrict__ nlist) {
  if (*nlist == 0) return;    // empty pixel list: k_exact_syrk wrote nothing
  const size_t total = (size_t)N * (N + 1) / 2 + N;
  for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (size_t)gridDim.x * blockDim.x) {
    int i, j;
    bool rhs = false;
    if (e < (size_t)N * (N + 1) / 2) {   // lower-triangle entry (i >= j)
      i = (int)((sqrt(8.0 * (double)e + 1.0) - 1.0) * 0.5);
      while ((size_t)(i + 1) * (i + 2) / 2 <= e) ++i;
      while ((size_t)i * (i + 1) / 2 > e) --i;
      j = (int)(e - (size_t)i * (i + 1) / 2);
    } else {
      rhs = true;
      i = N;
      j = (int)(e - (size_t)N * (N + 1) / 2);
    }
    const int ti = i / EX_T, tj = j / EX_T;
    const size_t loc = ((size_t)(ti * (ti + 1) / 2 + tj) * EX_T + (i % EX_T)) * EX_T + (j % EX_T);
    double s = 0.0;
    for (int ks = 0; ks < KSplit; ++ks) s += Cpart[(size_t)ks * ntiles * EX_T * EX_T + loc];
    s *= sign;
    if (rhs) {
      b[j] += s;
    } else {
      A[(size_t)i * N + j] += s;
      if (i != j) A[(size_t)j * N + i] += s;
    }
  }
}

static int exact_ksplit(int ntiles, int num_sms) {   // every CTA of the cooperative grid must be resident
  int ks = num_sms / ntiles;
  if (ks < 1) ks = 1;
  if (ks > 16) ks = 16;
  return ks;
}

// the rank-K update keeps one 128 x 128 tile of the lower triangle per CTA of a cooperative launch: N + 1 <= 16 * 128
// on a 148-SM device (w <= 5 always fits; w = 8 with DK = 2 is the largest kernel model that does)
bool sfft_exact_supported(int N, int num_sms) {
  const int ntb = (N + 1 + EX_T - 1) / EX_T;
  return ntb * (ntb + 1) / 2 <= num_sms;
}

size_t sfft_exact_scratch_bytes(int N, int num_sms) {
  if (!sfft_exact_supported(N, num_sms)) return 256;
  const int ntb = (N + 1 + EX_T - 1) / EX_T, ntiles = ntb * (ntb + 1) / 2;
  return (size_t)16 * ntiles * EX_T * EX_T * sizeof(double);
}

size_t sfft_exact_rows_bytes(int N, int num_sms) {
  if (!sfft_exact_supported(N, num_sms)) return 256;
  const int ntb = (N + 1 + EX_T - 1) / EX_T;
  return (size_t)EX_KC * ntb * EX_T * sizeof(double);
}

void sfft_launch_mk_scan(const int* cnt, int* off, int H, cudaStream_t st) { k_mk_scan<<<1, 1024, 0, st>>>(cnt, off, H); }

// rank-K update over one ordered pixel list: A, b += sign * sum_{x in list} g(x) [g(x); S(x)]^T
sfft_status sfft_launch_exact_syrk(sfft_plan* p, const double* R, const double* S, const int* list, const int* off,
                                   double* A, double* b, double sign, cudaStream_t st, int* nl) {
  const int H = p->H, W = p->W;
  ExactParams P;
  P.R = R; P.S = S; P.list = list; P.off = off; P.Cpart = p->exScratch;
  P.H = H; P.W = W; P.w = p->w; P.L = p->L; P.TK = p->TK; P.TB = p->TB; P.N = p->N;
  P.ntb = (p->N + 1 + EX_T - 1) / EX_T;
  P.log2W = p->log2NC + 1;
  const int ntiles = P.ntb * (P.ntb + 1) / 2;
  if (ntiles > p->num_sms) return SFFT_ERR_UNSUPPORTED;
  const int ks = exact_ksplit(ntiles, p->num_sms);
  P.KSplit = ks;
  P.Gm = p->exRows; P.bar = p->exBar;
  for (int t = 0; t < p->TK; ++t) { P.monoK[t][0] = p->monoK[t][0]; P.monoK[t][1] = p->monoK[t][1]; }
  for (int t = 0; t < p->TB; ++t) { P.monoB[t][0] = p->monoB[t][0]; P.monoB[t][1] = p->monoB[t][1]; }
  const size_t smem = (size_t)2 * 2 * EX_KS * EX_PITCH * sizeof(double);
  SFFT_CUDA_TRY(cudaFuncSetAttribute(k_exact_syrk, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  void* args[] = {(void*)&P};
  SFFT_CUDA_TRY(cudaLaunchCooperativeKernel((const void*)k_exact_syrk, dim3(ntiles, ks), dim3(EX_TH), args, smem, st));
  k_exact_apply<<<p->num_sms * 4, 256, 0, st>>>(p->exScratch, A, b, p->N, ntiles, ks, sign, off + H);
  SFFT_LAUNCH_CHECK();
  *nl += 2;
  return SFFT_OK;
}
