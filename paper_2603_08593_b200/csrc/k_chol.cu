// Blocked fp64 Cholesky solve of the normal equations (north_star subsystem (5)).
//
// Right-looking blocked factorisation A = Lc Lc^T, block size NB = 32, on the augmented matrix
// [A b; b^T .]: carrying b as row N through the panel solves yields z = Lc^-1 b for free (the
// forward substitution), so only the back substitution Lc^T c = z remains.
//   k_chol_load   : copy the lower triangle of A and b into the workspace (inputs stay untouched)
//   k_chol_panel  : every CTA factors the 32x32 diagonal block in shared memory (redundantly, which
//                   saves a launch), then solves its rows of the panel X Lkk^T = A_ik, one row per
//                   thread, by substitution (backward stable; no explicit block inverse)
//   k_chol_update : trailing update A22 -= L21 L21^T on 32x32 tiles of the lower triangle
//   k_chol_back   : one CTA, blocked back substitution with the stored diagonal factors
// info: 0, or the 1-based order of the first non-positive leading minor (no pivoting, no
// regularisation: DESIGN.md reading A9).
#include "sfft_common.cuh"

#define CH_NB 32

__global__ void __launch_bounds__(256) k_chol_load(const double* __restrict__ A,
                                                    const double* __restrict__ b, double* Lw, int N,
                                                    int ld, int* info) {
  const size_t total = (size_t)(N + 1) * N;
  if (blockIdx.x == 0 && threadIdx.x == 0 && info) *info = 0;
  for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < total;
       e += (size_t)gridDim.x * blockDim.x) {
    const int i = (int)(e / N), j = (int)(e - (size_t)i * N);
    if (i == N) Lw[(size_t)N * ld + j] = b[j];
    else if (j <= i) Lw[(size_t)i * ld + j] = A[e];
  }
}

__global__ void __launch_bounds__(128) k_chol_panel(double* Lw, double* Ldiag, int N, int ld, int k0,
                                                     int* info) {
  __shared__ double sd[CH_NB][CH_NB + 1];
  const int tid = threadIdx.x;
  const int nb = min(CH_NB, N - k0);
  for (int e = tid; e < CH_NB * CH_NB; e += 128) {
    const int i = e / CH_NB, j = e % CH_NB;
    sd[i][j] = (i < nb && j <= i) ? Lw[(size_t)(k0 + i) * ld + k0 + j] : (i == j ? 1.0 : 0.0);
  }
  __syncthreads();
  for (int k = 0; k < nb; ++k) {
    if (tid == 0) {
      double d = sd[k][k];
      if (!(d > 0.0)) {
        if (blockIdx.x == 0 && info) atomicCAS(info, 0, k0 + k + 1);
        d = 1.0;
      }
      sd[k][k] = sqrt(d);
    }
    __syncthreads();
    if (tid > k && tid < nb) sd[tid][k] /= sd[k][k];
    __syncthreads();
    // trailing update of the block: elements (i,j), k < j <= i < nb
    for (int e = tid; e < CH_NB * CH_NB; e += 128) {
      const int i = e / CH_NB, j = e % CH_NB;
      if (j > k && j <= i && i < nb) sd[i][j] = fma(-sd[i][k], sd[j][k], sd[i][j]);
    }
    __syncthreads();
  }
  if (blockIdx.x == 0) {
    double* dst = Ldiag + (size_t)(k0 / CH_NB) * CH_NB * CH_NB;
    for (int e = tid; e < CH_NB * CH_NB; e += 128) dst[e] = sd[e / CH_NB][e % CH_NB];
  }
  // panel rows below the diagonal block (including the rhs row N): one row per thread
  const int row = k0 + nb + blockIdx.x * 128 + tid;
  if (row <= N) {
    double x[CH_NB];
    double* src = Lw + (size_t)row * ld + k0;
#pragma unroll
    for (int j = 0; j < CH_NB; ++j) x[j] = (j < nb) ? src[j] : 0.0;
#pragma unroll
    for (int j = 0; j < CH_NB; ++j) {
      double a = x[j];
#pragma unroll
      for (int m = 0; m < j; ++m) a = fma(-x[m], sd[j][m], a);
      x[j] = a / sd[j][j];
    }
#pragma unroll
    for (int j = 0; j < CH_NB; ++j)
      if (j < nb) src[j] = x[j];
  }
}

__global__ void __launch_bounds__(256) k_chol_update(double* Lw, int N, int ld, int k0) {
  // tile (ti, tj), tj <= ti, of the trailing matrix starting at r0 = k0 + NB
  const int r0 = k0 + CH_NB;
  const int ti = blockIdx.y, tj = blockIdx.x;
  if (tj > ti) return;
  __shared__ double pi[CH_NB][CH_NB + 1], pj[CH_NB][CH_NB + 1];
  const int tid = threadIdx.x;
  for (int e = tid; e < CH_NB * CH_NB; e += 256) {
    const int r = e / CH_NB, m = e % CH_NB;
    const int gi = r0 + ti * CH_NB + r, gj = r0 + tj * CH_NB + r;
    pi[r][m] = (gi <= N) ? Lw[(size_t)gi * ld + k0 + m] : 0.0;
    pj[r][m] = (gj < N) ? Lw[(size_t)gj * ld + k0 + m] : 0.0;
  }
  __syncthreads();
  const int c = tid & 31, rb = tid >> 5;  // 8 row groups x 32 columns; 4 rows each
#pragma unroll
  for (int rr = 0; rr < 4; ++rr) {
    const int r = rb * 4 + rr;
    const int gi = r0 + ti * CH_NB + r, gj = r0 + tj * CH_NB + c;
    if (gi <= N && gj < N && gj <= gi) {
      double a = 0.0;
#pragma unroll
      for (int m = 0; m < CH_NB; ++m) a = fma(pi[r][m], pj[c][m], a);
      Lw[(size_t)gi * ld + gj] -= a;
    }
  }
}

__global__ void __launch_bounds__(1024) k_chol_back(const double* __restrict__ Lw,
                                                     const double* __restrict__ Ldiag, double* c,
                                                     int N, int ld) {
  extern __shared__ double sm[];
  double* r = sm;             // N running right-hand side
  double* ld_s = sm + N;      // 32 x 33 diagonal factor
  double* cb = ld_s + CH_NB * (CH_NB + 1);  // 32 solved values of the current block
  const int tid = threadIdx.x;
  for (int j = tid; j < N; j += 1024) r[j] = Lw[(size_t)N * ld + j];
  const int nblk = (N + CH_NB - 1) / CH_NB;
  for (int kb = nblk - 1; kb >= 0; --kb) {
    const int k0 = kb * CH_NB;
    const int nb = min(CH_NB, N - k0);
    __syncthreads();
    for (int e = tid; e < CH_NB * CH_NB; e += 1024)
      ld_s[(e / CH_NB) * (CH_NB + 1) + (e % CH_NB)] = Ldiag[(size_t)kb * CH_NB * CH_NB + e];
    __syncthreads();
    if (tid < 32) {
      // Lkk^T x = r_k: lane m holds r_m; columns solved from the last to the first
      double rm = (tid < nb) ? r[k0 + tid] : 0.0;
      for (int j = nb - 1; j >= 0; --j) {
        const double rj = __shfl_sync(0xffffffffu, rm, j);
        const double xj = rj / ld_s[j * (CH_NB + 1) + j];
        if (tid == j) rm = xj;
        else if (tid < j) rm = fma(-ld_s[j * (CH_NB + 1) + tid], xj, rm);
      }
      if (tid < nb) {
        cb[tid] = rm;
        c[k0 + tid] = rm;
      }
    }
    __syncthreads();
    // r[j] -= sum_i L[k0+i][j] x_i for all j < k0 (coalesced along j)
    for (int j = tid; j < k0; j += 1024) {
      double a = r[j];
#pragma unroll 8
      for (int i = 0; i < nb; ++i) a = fma(-Lw[(size_t)(k0 + i) * ld + j], cb[i], a);
      r[j] = a;
    }
  }
}

sfft_status sfft_launch_solve(sfft_plan* p, const double* A, const double* b, double* c, int* info,
                              cudaStream_t st, int* nl) {
  const int N = p->N, ld = p->ldL;
  k_chol_load<<<148 * 4, 256, 0, st>>>(A, b, p->Lw, N, ld, info);
  SFFT_LAUNCH_CHECK();
  ++*nl;
  for (int k0 = 0; k0 < N; k0 += CH_NB) {
    const int nb = (N - k0) < CH_NB ? (N - k0) : CH_NB;
    const int rows_below = N + 1 - (k0 + nb);  // includes the rhs row
    const int gp = rows_below > 0 ? (rows_below + 127) / 128 : 1;
    k_chol_panel<<<gp, 128, 0, st>>>(p->Lw, p->Ldiag, N, ld, k0, info);
    SFFT_LAUNCH_CHECK();
    ++*nl;
    if (k0 + CH_NB < N) {
      const int nt = (N + 1 - (k0 + CH_NB) + CH_NB - 1) / CH_NB;
      dim3 g(nt, nt);
      k_chol_update<<<g, 256, 0, st>>>(p->Lw, N, ld, k0);
      SFFT_LAUNCH_CHECK();
      ++*nl;
    } else if (k0 + nb < N + 1 && k0 + CH_NB >= N) {
      // last panel: nothing but the rhs row's own (unused) diagonal entry remains
    }
  }
  const size_t smem = ((size_t)N + CH_NB * (CH_NB + 1) + CH_NB) * sizeof(double);
  SFFT_CUDA_TRY(cudaFuncSetAttribute(k_chol_back, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  k_chol_back<<<1, 1024, smem, st>>>(p->Lw, p->Ldiag, c, N, ld);
  SFFT_LAUNCH_CHECK();
  ++*nl;
  return SFFT_OK;
}
