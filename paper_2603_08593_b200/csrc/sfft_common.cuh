// Common definitions for the sm_100a SFFT kernels: plan layout, complex helpers, launch checks.
// Conventions follow include/sfft.h.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/sfft.h"

#define SFFT_MAX_DEG 3
#define SFFT_MAX_T 10     // (3+1)(3+2)/2 monomials of degree <= 3
#define SFFT_MAX_W 15
#define SFFT_PITCH_PAD 16   // spectrum row pitch = W/2 + 16 complex (column W/2 = Nyquist; a 16-column tile at W/2 stays in the row)
#define SFFT_CR_CT 16        // k_cross: columns per CTA
#define SFFT_CR_GP 21        // k_cross: pairs per CTA (threads = SFFT_CR_GP * SFFT_CR_CT)
#define SFFT_CR_MAXSPEC 24   // k_cross: spectra a group may stage
#ifndef SFFT_KB_NBLK
#define SFFT_KB_NBLK 296     // x-CTAs of the kernel-background correction kernel (2 per SM)
#endif
#ifndef SFFT_T_G
#define SFFT_T_G 4          // fused path: rows per group of the row-spectra layout T[img][y/G][kx][y%G] (2, 4 and 8 measured: 4 is best)
#endif
#define SFFT_XS_MAXT 32     // exact objective, structured part (k_exact_strips.cu): most fully masked lines per direction,
#define SFFT_XS_MAXS 64     //   most distinct source lines,
#define SFFT_XS_MAXW 5      //   largest kernel half-width it is compiled for
#define SFFT_NSTAGE 10     // see sfft_profile_read in include/sfft.h
#define SFFT_PROF_MAX 512

typedef double2 cplx;

__host__ __device__ __forceinline__ cplx cmake(double a, double b) { return make_double2(a, b); }
__device__ __forceinline__ cplx cadd(cplx a, cplx b) { return cmake(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ cplx csub(cplx a, cplx b) { return cmake(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ cplx cconj(cplx a) { return cmake(a.x, -a.y); }
__device__ __forceinline__ cplx cscale(cplx a, double s) { return cmake(a.x * s, a.y * s); }
// a*b
__device__ __forceinline__ cplx cmul(cplx a, cplx b) {
  return cmake(fma(a.x, b.x, -(a.y * b.y)), fma(a.x, b.y, a.y * b.x));
}
// conj(a)*b
__device__ __forceinline__ cplx cmulc(cplx a, cplx b) {
  return cmake(fma(a.x, b.x, a.y * b.y), fma(a.x, b.y, -(a.y * b.x)));
}
// acc += a*b
__device__ __forceinline__ void cfma(cplx& acc, cplx a, cplx b) {
  acc.x = fma(a.x, b.x, acc.x);
  acc.x = fma(-a.y, b.y, acc.x);
  acc.y = fma(a.x, b.y, acc.y);
  acc.y = fma(a.y, b.x, acc.y);
}
// acc += conj(a)*b
__device__ __forceinline__ void cfmac(cplx& acc, cplx a, cplx b) {
  acc.x = fma(a.x, b.x, acc.x);
  acc.x = fma(a.y, b.y, acc.x);
  acc.y = fma(a.x, b.y, acc.y);
  acc.y = fma(-a.y, b.x, acc.y);
}
// multiply by +i / -i
__device__ __forceinline__ cplx cmul_pi(cplx a) { return cmake(-a.y, a.x); }
__device__ __forceinline__ cplx cmul_mi(cplx a) { return cmake(a.y, -a.x); }

__device__ __forceinline__ cplx ldg2(const cplx* p) { return __ldg(p); }

__device__ __forceinline__ double ipow(double x, int n) {
  double r = 1.0;
  for (int i = 0; i < n; ++i) r *= x;
  return r;
}

// A cross-correlation pair: spectra indices into the plan's spectrum array and its lag half-range.
struct PairDesc {
  int fa;   // spectrum index of f  (conj side)
  int fb;   // spectrum index of g
  int D;    // lags needed: dy,dx in [-D, D]
};

// A group of pairs handled by one k_cross CTA: the spectra it stages and, per pair, the local slots
// of its two spectra and its row block in Y.  All pairs of a group share the lag half-range D.
struct CrossGroup {
  int ns, np, D, pad;
  int spec[SFFT_CR_MAXSPEC];
  int la[SFFT_CR_GP], lb[SFFT_CR_GP];
  int pair[SFFT_CR_GP];
};

struct sfft_plan {
  int H, W, w, DK, DB;
  int L, TK, TB, N;
  int NC;        // W/2
  int pitch;     // spectrum row pitch (complex elements) = NC + SFFT_PITCH_PAD
  int log2H, log2NC;
  int nRowImg;   // forward row-pass images in build: R~ xi^p (DK+1), S~ (1)
  int nSpec;     // spectra: TK + 1  (the kernel-background block needs none, see k_kb.cu)
  int nPair;     // TK(TK+1)/2 + TK
  int Dmax;      // 2w
  int nLag;      // 2*Dmax+1
  int monoK[SFFT_MAX_T][2], monoB[SFFT_MAX_T][2];
  int nMomA;     // 2*DB+1 row moments  sum_x m xi^a
  int nMomS;     // DB+1 row moments     sum_x m xi^p S
  int nMomR;     // DK+DB+1 row moments  sum_x m xi^a R
  double fullA[2 * SFFT_MAX_DEG + 1];   // sum_x xi(x)^a over one whole row (long double on the host)

  // device tables
  cplx* twPNC;   // per-pass FFT twiddle tables for length NC (fft_smem.cuh)
  cplx* twPH;    // per-pass FFT twiddle tables for length H
  cplx* tw128;   // e^{-2 pi i m/128}: block transforms of the blocked column/cross kernel (k_colb.cu)
  int fused;     // 1: k_colb replaces k_col_fwd + k_cross (H in {1024,2048,4096}, <= 32 pairs)
  int nPart;     // partial lag-row sets in Y (1 on both paths)
  int pitchT;    // row pitch of T on the generic build path (NC packed); the fused path is column-major
  cplx* twW;     // e^{-2 pi i m / W},  m in [0, W)
  cplx* twH;     // e^{-2 pi i m / H},  m in [0, H)
  PairDesc* d_pairs;
  PairDesc* h_pairs;
  CrossGroup* d_groups;   // kernel-kernel groups first, then the D = w groups
  int nGroupKK, nGroupKO, maxnsKK, maxnsKO;

  // device scratch
  cplx* T;       // row-pass output  [nRowImg][H][NC]   (packed: column 0 = DC + i Nyquist)
  cplx* F;       // spectra          [nSpec][H][pitch]  (column NC = Nyquist)
  cplx* Y;       // lag rows         [nPair][nLag][pitch]
  double* Cmap;  // lag windows      [nPair][nLag][nLag]
  double* rowMom;   // [nMomA + nMomS + nMomR][H]
  double* mom;      // [nMomA^2] mask moments, [TB] background rhs, [nMomR^2] moments of m R
  // kernel-background block without transforms (k_kb.cu): special target pixels (masked, or within
  // w of an edge), their per-row counts/offsets, per-CTA partial corrections and the reduced ones
  int* spCount;     // [H]
  int* spOff;       // [H + 1]   exclusive scan; spOff[H] = number of special pixels
  int* spList;      // [H*W]     y*W + x, bit 31 set when the pixel is masked
  int* fmFlag;      // [H]       1 if every pixel of the row is masked (such rows are not listed)
  int* fmList;      // [H + 1]   number of fully masked rows, then the rows in ascending order
  double* kbPart;   // [KB_NBLK][L*TK*TB]
  double* kbCorr;   // [L*TK*TB]
  double* kbStrip;  // [L*TK*TB] part of the fully masked target rows (from row moments)
  double* Lw;       // Cholesky workspace (N+1) x ldL
  double* exScratch; // sfft_build_system_exact: partial tiles of the masked pixels' rank-K update
  double* exRows;    //   generated design-matrix rows of one chunk of masked pixels (allocated on first use)
  unsigned* exBar;   //   grid-barrier counters of k_exact_syrk
  // fully masked rows / columns of the exact objective (k_exact_strips.cu)
  void* xsPlan;             // 2 x XsPlan
  int* xsColCnt;            // [W]
  unsigned char* xsRowFull; // [H]
  unsigned char* xsColFull; // [W]
  int* xsSrcIdxY;           // [H]
  int* xsSrcIdxX;           // [W]
  double* xsZ;              // strips
  double* xsQ;              // strip correlations
  int* xsCnt;               // [H]     corner list: per-row counts,
  int* xsOff;               // [H + 1] offsets,
  int* xsList;              // [XS_MAXT^2] pixels
  int cholMaxCtas;   // cap on the CTAs of k_chol_fused (0 = one per SM); see sfft_plan_set_solve_ctas
  double* mtA;       // sfft_multi_template_difference: normal matrix and right-hand side of the current template
  double* mtB;
  unsigned* cholBar; // grid-barrier counters of k_chol_fused (arrivals, finished CTAs)
  cplx* Etab;       // subtract: E[TK][2w+1][NC]
  cplx* Mhat;       // subtract: mixed row spectra [H][NC]
  int ldL;
  size_t ws_bytes;
  int launches[3];
  int num_sms;
  // plan-owned side stream: stages of one call that do not depend on each other run concurrently
  // (forked from and joined back into the caller stream with events; no host synchronisation)
  cudaStream_t side;
  cudaEvent_t evFork, evJoin, evRow, evPrep;
  // sfft_multi_template_difference_plans: the chains a helper plan runs go to its own work stream
  cudaStream_t work;
  cudaEvent_t evWork, evBuilt;
  // sfft_subtract_prepare: the row spectra of xi^p R for the next sfft_subtract are already in T
  const double* prepR;
  int prepValid;
  // optional per-stage CUDA-event timing (sfft_profile_*): events are recorded on the caller
  // stream around each stage; nothing synchronises until sfft_profile_read.
  int prof_on;
  int prof_n;                       // recorded (stage, e0, e1) triples awaiting a read
  int prof_stage[SFFT_PROF_MAX];
  cudaEvent_t prof_ev[2 * SFFT_PROF_MAX];
  double prof_ms[SFFT_NSTAGE];
  int prof_cnt[SFFT_NSTAGE];
};

struct ProfScope {  // RAII: record an event pair around one stage when profiling is on
  sfft_plan* p; cudaStream_t st; int slot;
  ProfScope(sfft_plan* p_, int stage, cudaStream_t st_) : p(p_), st(st_), slot(-1) {
    if (p->prof_on && p->prof_n < SFFT_PROF_MAX) {
      slot = p->prof_n++;
      p->prof_stage[slot] = stage;
      cudaEventRecord(p->prof_ev[2 * slot], st);
    }
  }
  ~ProfScope() { if (slot >= 0) cudaEventRecord(p->prof_ev[2 * slot + 1], st); }
};

#define SFFT_CUDA_TRY(expr)                          \
  do {                                               \
    cudaError_t _e = (expr);                         \
    if (_e != cudaSuccess) return SFFT_ERR_CUDA;     \
  } while (0)

#define SFFT_LAUNCH_CHECK()                          \
  do {                                               \
    if (cudaPeekAtLastError() != cudaSuccess) {      \
      cudaGetLastError();                            \
      return SFFT_ERR_CUDA;                          \
    }                                                \
  } while (0)

// SM count of the current device (cached; 148 on B200), for the plan-less calls' grid sizes
inline int sfft_device_sms() {
  static int n = 0;
  if (n == 0) {
    int dev = 0, v = 0;
    if (cudaGetDevice(&dev) == cudaSuccess &&
        cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && v > 0) n = v;
    else { cudaGetLastError(); return 148; }
  }
  return n;
}

// ---- stage entry points implemented in the k_*.cu files (host functions) ----------------------
// build = true: images m xi^p R (p <= DK) and m S with the fused row moments; false: xi^p R only
sfft_status sfft_launch_row_fwd(sfft_plan* p, const double* R, const double* S,
                                const unsigned char* mask, bool build, cplx* Tout, int pitchT, bool packed,
                                bool colT, cudaStream_t st, int* nl);
sfft_status sfft_launch_col_fwd(sfft_plan* p, cudaStream_t st, int* nl);
sfft_status sfft_launch_cross(sfft_plan* p, cudaStream_t st, int* nl);
sfft_status sfft_launch_colx(sfft_plan* p, cudaStream_t st, int* nl);
bool sfft_exact_supported(int N, int num_sms);
size_t sfft_exact_scratch_bytes(int N, int num_sms);
size_t sfft_exact_rows_bytes(int N, int num_sms);
size_t sfft_xs_plan_bytes();
size_t sfft_xs_strip_bytes(int H, int W);
size_t sfft_xs_q_bytes();
sfft_status sfft_launch_exact_update(sfft_plan* p, const double* R, const double* S, const unsigned char* mask,
                                     double* A, double* b, cudaStream_t st, int* nl);
bool sfft_colx_supported(int H, int nPair, int Dmax);
sfft_status sfft_launch_kb(sfft_plan* p, const double* R, const unsigned char* mask, cudaStream_t st, int* nl);
sfft_status sfft_launch_moments(sfft_plan* p, cudaStream_t st, int* nl);
sfft_status sfft_launch_lag_gather(sfft_plan* p, double* A, double* b, cudaStream_t st, int* nl);
sfft_status sfft_launch_solve(sfft_plan* p, const double* A, const double* b, double* c, int* info,
                              cudaStream_t st, int* nl);
sfft_status sfft_launch_subtract(sfft_plan* p, const double* R, const double* S, const double* c,
                                 double* D, cudaStream_t st, int* nl);
sfft_status sfft_launch_subtract_rows(sfft_plan* p, const double* R, cudaStream_t st, int* nl);
sfft_status sfft_run_probe(int kind, int iters, double* tflops, double* ms, cudaStream_t st);
