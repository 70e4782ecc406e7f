// C ABI of libsfft.so (include/sfft.h): plan management and stage scheduling on the caller stream.
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <new>
#include <vector>

#include "fft_smem.cuh"

static bool is_pow2(int v) { return v > 0 && (v & (v - 1)) == 0; }
static int ilog2(int v) { int l = 0; while ((1 << l) < v) ++l; return l; }

static int fill_monomials(int D, int (*m)[2]) {
  int n = 0;
  for (int d = 0; d <= D; ++d)
    for (int q = 0; q <= d; ++q) { m[n][0] = d - q; m[n][1] = q; ++n; }
  return n;
}

static cudaError_t upload_twiddles(cplx** dst, int n) {
  std::vector<cplx> h(n);
  const long double twopi = 6.283185307179586476925286766559005768L;
  for (int m = 0; m < n; ++m) {
    // exact values on the axes and diagonals, long double elsewhere (rounded once to double)
    const long double ang = -twopi * (long double)m / (long double)n;
    long double c = cosl(ang), s = sinl(ang);
    if ((4 * m) % n == 0) {
      const int quad = (4 * m) / n;  // multiples of pi/2
      c = (quad == 0) ? 1.0L : (quad == 2 ? -1.0L : 0.0L);
      s = (quad == 1) ? -1.0L : (quad == 3 ? 1.0L : 0.0L);
    }
    h[m] = cmake((double)c, (double)s);
  }
  cudaError_t e = cudaMalloc((void**)dst, sizeof(cplx) * (size_t)n);
  if (e != cudaSuccess) return e;
  return cudaMemcpy(*dst, h.data(), sizeof(cplx) * (size_t)n, cudaMemcpyHostToDevice);
}

// long-double e^{-2 pi i num/den}, exact on the axes, rounded once to double
static cplx unit_root(long long num, long long den) {
  const long double twopi = 6.283185307179586476925286766559005768L;
  num %= den;
  if ((4 * num) % den == 0) {
    const int quad = (int)((4 * num) / den);
    return cmake(quad == 0 ? 1.0 : (quad == 2 ? -1.0 : 0.0), quad == 1 ? -1.0 : (quad == 3 ? 1.0 : 0.0));
  }
  const long double ang = -twopi * (long double)num / (long double)den;
  return cmake((double)cosl(ang), (double)sinl(ang));
}

// Per-pass twiddle tables of the length-n FFT (layout: fft_smem.cuh): pass i >= 1 with radix R and
// stride NS stores exp(-2 pi i r k/(NS R)) at off_i + (r-1)*NS + k.
static cudaError_t upload_pass_tables(cplx** dst, int n) {
  std::vector<cplx> h(fft_pass_table_size(n), cmake(1.0, 0.0));
  for (int pass = 1; pass < fft_num_passes(n); ++pass) {
    const int R = fft_radix(n, pass), NS = fft_pass_ns(n, pass), off = fft_tw_off(n, pass);
    for (int r = 1; r < R; ++r)
      for (int k = 0; k < NS; ++k) h[off + (r - 1) * NS + k] = unit_root((long long)r * k, (long long)NS * R);
  }
  cudaError_t e = cudaMalloc((void**)dst, sizeof(cplx) * h.size());
  if (e != cudaSuccess) return e;
  return cudaMemcpy(*dst, h.data(), sizeof(cplx) * h.size(), cudaMemcpyHostToDevice);
}

static void plan_free(sfft_plan* p) {
  if (!p) return;
  cudaFree(p->tw128);
  cudaFree(p->twPNC); cudaFree(p->twPH); cudaFree(p->twW); cudaFree(p->twH); cudaFree(p->d_pairs); cudaFree(p->d_groups);
  cudaFree(p->T); cudaFree(p->F); cudaFree(p->Y); cudaFree(p->Cmap); cudaFree(p->rowMom);
  cudaFree(p->mom); cudaFree(p->spCount); cudaFree(p->spOff); cudaFree(p->spList); cudaFree(p->fmFlag); cudaFree(p->fmList); cudaFree(p->kbPart); cudaFree(p->kbCorr); cudaFree(p->kbStrip); cudaFree(p->Lw); cudaFree(p->exScratch); cudaFree(p->exRows); cudaFree(p->exBar); cudaFree(p->xsPlan); cudaFree(p->xsColCnt); cudaFree(p->xsRowFull); cudaFree(p->xsColFull); cudaFree(p->xsSrcIdxY); cudaFree(p->xsSrcIdxX); cudaFree(p->xsZ); cudaFree(p->xsQ); cudaFree(p->xsCnt); cudaFree(p->xsOff); cudaFree(p->xsList); cudaFree(p->cholBar); cudaFree(p->mtA); cudaFree(p->mtB); cudaFree(p->Etab); cudaFree(p->Mhat);
  free(p->h_pairs);
  if (p->side) cudaStreamDestroy(p->side);
  if (p->work) cudaStreamDestroy(p->work);
  if (p->evWork) cudaEventDestroy(p->evWork);
  if (p->evBuilt) cudaEventDestroy(p->evBuilt);
  if (p->evFork) cudaEventDestroy(p->evFork);
  if (p->evJoin) cudaEventDestroy(p->evJoin);
  if (p->evRow) cudaEventDestroy(p->evRow);
  if (p->evPrep) cudaEventDestroy(p->evPrep);
  for (int i = 0; i < 2 * SFFT_PROF_MAX; ++i) if (p->prof_ev[i]) cudaEventDestroy(p->prof_ev[i]);
  delete p;
}

static bool aligned16(const void* q) { return (((uintptr_t)q) & 15) == 0; }

extern "C" {

const char* sfft_version(void) { return "sfft-b200 0.1 (sm_100a)"; }

const char* sfft_status_string(sfft_status s) {
  switch (s) {
    case SFFT_OK: return "SFFT_OK";
    case SFFT_ERR_INVALID_ARG: return "SFFT_ERR_INVALID_ARG";
    case SFFT_ERR_UNSUPPORTED: return "SFFT_ERR_UNSUPPORTED";
    case SFFT_ERR_ALLOC: return "SFFT_ERR_ALLOC";
    case SFFT_ERR_CUDA: return "SFFT_ERR_CUDA";
    default: return "SFFT_ERR_UNKNOWN";
  }
}

sfft_status sfft_plan_create(sfft_plan** out, int H, int W, int w, int DK, int DB) {
  if (!out) return SFFT_ERR_INVALID_ARG;
  *out = nullptr;
  if (!is_pow2(H) || !is_pow2(W) || H < 16 || W < 16 || H > 4096 || W > 4096) return SFFT_ERR_UNSUPPORTED;
  if (w < 0 || w > SFFT_MAX_W || 4 * w + 1 > (H < W ? H : W)) return SFFT_ERR_UNSUPPORTED;
  if (DK < 0 || DK > SFFT_MAX_DEG || DB < 0 || DB > SFFT_MAX_DEG) return SFFT_ERR_UNSUPPORTED;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { cudaGetLastError(); return SFFT_ERR_CUDA; }

  sfft_plan* p = new (std::nothrow) sfft_plan;
  if (!p) return SFFT_ERR_ALLOC;
  memset(p, 0, sizeof(*p));
  p->H = H; p->W = W; p->w = w; p->DK = DK; p->DB = DB;
  p->L = (2 * w + 1) * (2 * w + 1);
  p->TK = fill_monomials(DK, p->monoK);
  p->TB = fill_monomials(DB, p->monoB);
  p->N = p->L * p->TK + p->TB;
  p->NC = W / 2;
  p->pitch = p->NC + SFFT_PITCH_PAD;
  p->log2H = ilog2(H); p->log2NC = ilog2(p->NC);
  p->nRowImg = (DK + 1) + 1;
  p->nSpec = p->TK + 1;
  p->nPair = p->TK * (p->TK + 1) / 2 + p->TK;
  p->Dmax = 2 * w;
  p->nLag = 2 * p->Dmax + 1;
  p->nMomA = 2 * DB + 1;
  p->nMomS = DB + 1;
  p->nMomR = DK + DB + 1;
  p->ldL = (p->N + 1 + 3) & ~3;
  p->fused = sfft_colx_supported(H, p->nPair, p->Dmax) ? 1 : 0;
  p->nPart = 1;
  p->pitchT = p->NC;
  for (int a = 0; a <= 2 * SFFT_MAX_DEG; ++a) {   // whole-row sums of xi^a (odd powers cancel exactly)
    long double acc = 0.0L;
    if ((a & 1) == 0)
      for (int x = 0; x < W; ++x) acc += powl((long double)(2 * x + 1 - W) / (long double)W, (long double)a);
    p->fullA[a] = (double)acc;
  }
  int dev = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&p->num_sms, cudaDevAttrMultiProcessorCount, dev);

  // pair list: kernel-kernel pairs (t <= t2) first, then (t,S) for each t
  p->h_pairs = (PairDesc*)malloc(sizeof(PairDesc) * p->nPair);
  if (!p->h_pairs) { plan_free(p); return SFFT_ERR_ALLOC; }
  int n = 0;
  for (int t = 0; t < p->TK; ++t)
    for (int t2 = t; t2 < p->TK; ++t2) { p->h_pairs[n].fa = t; p->h_pairs[n].fb = t2; p->h_pairs[n].D = 2 * w; ++n; }
  for (int t = 0; t < p->TK; ++t) {
    p->h_pairs[n].fa = t; p->h_pairs[n].fb = p->TK; p->h_pairs[n].D = w; ++n;
  }

  // k_cross groups: consecutive pairs (same D class) packed while the group holds <= SFFT_CR_GP
  // pairs and <= SFFT_CR_MAXSPEC distinct spectra
  std::vector<CrossGroup> groups;
  const int nKKpairs = p->TK * (p->TK + 1) / 2;
  for (int cls = 0; cls < 2; ++cls) {
    const int lo = cls == 0 ? 0 : nKKpairs, hi = cls == 0 ? nKKpairs : p->nPair;
    int maxns = 0, ng = 0;
    CrossGroup g; memset(&g, 0, sizeof(g));
    auto slot = [&](CrossGroup& gg, int spec) { for (int i = 0; i < gg.ns; ++i) if (gg.spec[i] == spec) return i; return -1; };
    auto flush = [&]() { if (g.np) { groups.push_back(g); if (g.ns > maxns) maxns = g.ns; ++ng; } memset(&g, 0, sizeof(g)); };
    for (int i = lo; i < hi; ++i) {
      const PairDesc& pd = p->h_pairs[i];
      int need = (slot(g, pd.fa) < 0) + (pd.fb != pd.fa && slot(g, pd.fb) < 0);
      if (g.np == SFFT_CR_GP || g.ns + need > SFFT_CR_MAXSPEC) flush();
      if (slot(g, pd.fa) < 0) g.spec[g.ns++] = pd.fa;
      if (slot(g, pd.fb) < 0) g.spec[g.ns++] = pd.fb;
      g.la[g.np] = slot(g, pd.fa); g.lb[g.np] = slot(g, pd.fb); g.pair[g.np] = i; g.D = pd.D; ++g.np;
    }
    flush();
    if (cls == 0) { p->nGroupKK = ng; p->maxnsKK = maxns; } else { p->nGroupKO = ng; p->maxnsKO = maxns; }
  }

  int prLo = 0, prHi = 0;   // the side stream's small kernels take free slots ahead of the big grids
  cudaDeviceGetStreamPriorityRange(&prLo, &prHi);
  if (cudaStreamCreateWithPriority(&p->side, cudaStreamNonBlocking, prHi) != cudaSuccess ||
      cudaStreamCreateWithPriority(&p->work, cudaStreamNonBlocking, prLo) != cudaSuccess ||
      cudaEventCreateWithFlags(&p->evWork, cudaEventDisableTiming) != cudaSuccess ||
      cudaEventCreateWithFlags(&p->evBuilt, cudaEventDisableTiming) != cudaSuccess ||
      cudaEventCreateWithFlags(&p->evFork, cudaEventDisableTiming) != cudaSuccess ||
      cudaEventCreateWithFlags(&p->evJoin, cudaEventDisableTiming) != cudaSuccess ||
      cudaEventCreateWithFlags(&p->evRow, cudaEventDisableTiming) != cudaSuccess ||
      cudaEventCreateWithFlags(&p->evPrep, cudaEventDisableTiming) != cudaSuccess) {
    cudaGetLastError();
    plan_free(p);
    return SFFT_ERR_CUDA;
  }
  size_t ws = 0;
  bool ok = true;
  auto dalloc = [&](void** ptr, size_t bytes) {
    if (!ok) return;
    if (cudaMalloc(ptr, bytes) != cudaSuccess) { cudaGetLastError(); ok = false; *ptr = nullptr; return; }
    ws += bytes;
  };
  const size_t HN = (size_t)H * p->NC, HP = (size_t)H * p->pitch;
  // fused path: column-major T[img][NC+1][H]; subtract always uses row-major packed [DK+1][H][NC]
  size_t Tbytes = sizeof(cplx) * (size_t)H * p->pitchT * p->nRowImg;
  if (p->fused) Tbytes = sizeof(cplx) * (size_t)H * (p->NC + 1) * p->nRowImg;
  const size_t Fbytes = p->fused ? 256 : sizeof(cplx) * HP * p->nSpec;   // no spectra in HBM on the fused path
  const size_t Ybytes = sizeof(cplx) * (size_t)p->nPart * p->nPair * p->nLag * p->pitch;
  dalloc((void**)&p->T, Tbytes);
  dalloc((void**)&p->F, Fbytes);
  dalloc((void**)&p->Y, Ybytes);
  dalloc((void**)&p->Cmap, sizeof(double) * (size_t)p->nPair * p->nLag * p->nLag);
  dalloc((void**)&p->rowMom, sizeof(double) * (size_t)(p->nMomA + p->nMomS + p->nMomR) * H);
  dalloc((void**)&p->mom, sizeof(double) * (size_t)(p->nMomA * p->nMomA + p->TB + p->nMomR * p->nMomR));
  {
    const int nsub = 128 / p->L > 0 ? 128 / p->L : 1;
    dalloc((void**)&p->spCount, sizeof(int) * (size_t)H);
    dalloc((void**)&p->spOff, sizeof(int) * (size_t)(H + 1));
    dalloc((void**)&p->spList, sizeof(int) * (size_t)H * W);
    dalloc((void**)&p->fmFlag, sizeof(int) * (size_t)H);
    dalloc((void**)&p->fmList, sizeof(int) * (size_t)(H + 1));
    dalloc((void**)&p->kbPart, sizeof(double) * (size_t)SFFT_KB_NBLK * nsub * p->TK * p->L * p->TB);
    dalloc((void**)&p->kbCorr, sizeof(double) * (size_t)p->TK * p->L * p->TB);
    dalloc((void**)&p->kbStrip, sizeof(double) * (size_t)p->TK * p->L * p->TB);
  }
  dalloc((void**)&p->exScratch, sfft_exact_scratch_bytes(p->N, p->num_sms));
  dalloc((void**)&p->exRows, sfft_exact_rows_bytes(p->N, p->num_sms));   // here, so that no hot call ever allocates
  dalloc((void**)&p->exBar, 2 * sizeof(unsigned));
  dalloc((void**)&p->xsPlan, sfft_xs_plan_bytes());
  dalloc((void**)&p->xsColCnt, sizeof(int) * (size_t)W);
  dalloc((void**)&p->xsRowFull, (size_t)H);
  dalloc((void**)&p->xsColFull, (size_t)W);
  dalloc((void**)&p->xsSrcIdxY, sizeof(int) * (size_t)H);
  dalloc((void**)&p->xsSrcIdxX, sizeof(int) * (size_t)W);
  dalloc((void**)&p->xsZ, sfft_xs_strip_bytes(H, W));
  dalloc((void**)&p->xsQ, sfft_xs_q_bytes());
  dalloc((void**)&p->xsCnt, sizeof(int) * (size_t)H);
  dalloc((void**)&p->xsOff, sizeof(int) * (size_t)(H + 1));
  dalloc((void**)&p->xsList, sizeof(int) * (size_t)SFFT_XS_MAXT * SFFT_XS_MAXT);
  dalloc((void**)&p->Lw, sizeof(double) * (size_t)(p->N + 1) * p->ldL);
  dalloc((void**)&p->cholBar, 2 * sizeof(unsigned));
  dalloc((void**)&p->mtA, sizeof(double) * (size_t)p->N * p->N);   // normal equations of the multi-template mode
  dalloc((void**)&p->mtB, sizeof(double) * (size_t)p->N);
  dalloc((void**)&p->Etab, sizeof(cplx) * (size_t)p->TK * (2 * w + 1) * p->NC);
  dalloc((void**)&p->Mhat, sizeof(cplx) * HN);
  dalloc((void**)&p->d_pairs, sizeof(PairDesc) * p->nPair);
  dalloc((void**)&p->d_groups, sizeof(CrossGroup) * groups.size());
  if (!ok) { plan_free(p); return SFFT_ERR_ALLOC; }
  if (p->fused && upload_twiddles(&p->tw128, 128) != cudaSuccess) {
    cudaGetLastError();
    plan_free(p);
    return SFFT_ERR_CUDA;
  }
  if (upload_pass_tables(&p->twPNC, p->NC) != cudaSuccess || upload_pass_tables(&p->twPH, H) != cudaSuccess || upload_twiddles(&p->twW, W) != cudaSuccess ||
      upload_twiddles(&p->twH, H) != cudaSuccess ||
      cudaMemcpy(p->d_pairs, p->h_pairs, sizeof(PairDesc) * p->nPair, cudaMemcpyHostToDevice) != cudaSuccess ||
      cudaMemcpy(p->d_groups, groups.data(), sizeof(CrossGroup) * groups.size(), cudaMemcpyHostToDevice) != cudaSuccess ||
      cudaMemset(p->exBar, 0, 2 * sizeof(unsigned)) != cudaSuccess ||
      cudaMemset(p->cholBar, 0, 2 * sizeof(unsigned)) != cudaSuccess ||
      cudaMemset(p->T, 0, Tbytes) != cudaSuccess ||
      cudaMemset(p->F, 0, Fbytes) != cudaSuccess ||
      cudaMemset(p->Y, 0, Ybytes) != cudaSuccess ||
      cudaMemset(p->Cmap, 0, sizeof(double) * (size_t)p->nPair * p->nLag * p->nLag) != cudaSuccess) {
    cudaGetLastError();
    plan_free(p);
    return SFFT_ERR_CUDA;
  }
  ws += sizeof(cplx) * (size_t)(fft_pass_table_size(p->NC) + fft_pass_table_size(H) + W + H);
  p->ws_bytes = ws;
  if (cudaDeviceSynchronize() != cudaSuccess) { cudaGetLastError(); plan_free(p); return SFFT_ERR_CUDA; }
  *out = p;
  return SFFT_OK;
}

sfft_status sfft_plan_destroy(sfft_plan* p) {
  if (!p) return SFFT_ERR_INVALID_ARG;
  plan_free(p);
  return SFFT_OK;
}

int sfft_num_coeffs(const sfft_plan* p) { return p ? p->N : -1; }
size_t sfft_workspace_bytes(const sfft_plan* p) { return p ? p->ws_bytes : 0; }

// A CUDA error left pending by earlier, unrelated work would be reported as a launch failure of this
// library (the launch checks peek at the last error): the hot calls refuse to start on top of one.
static bool cuda_error_pending() { return cudaPeekAtLastError() != cudaSuccess; }

// After the fork every failure path must join the side stream back into the caller stream: the side
// stream may still be reading the caller's R and mask, which the caller is free to reuse once the
// call has returned and its stream has drained.
static sfft_status fail_joined(sfft_plan* p, cudaStream_t st, sfft_status s) {
  if (cudaEventRecord(p->evJoin, p->side) == cudaSuccess) cudaStreamWaitEvent(st, p->evJoin, 0);
  cudaGetLastError();
  return s;
}

// reuseS: the row spectra and row moments of m S are already in the scratch (same S and mask as the
// previous build of this plan: the multi-template mode), only the R images are transformed
static sfft_status build_system_impl(sfft_plan* p, const double* R, const double* S, const unsigned char* mask,
                                     double* A, double* b, cudaStream_t st, bool reuseS = false) {
  int nl = 0;
  // the row-pass scratch is about to be overwritten: an unconsumed prepare finishes first, then is dropped
  if (p->prepValid) SFFT_CUDA_TRY(cudaStreamWaitEvent(st, p->evPrep, 0));
  p->prepValid = 0;
  // a1 + a2 (row pass): m xi^p R (p<=DK), m S, with the fused moment reductions
  // (sum m xi^a, sum m S xi^p, sum m R xi^a)
  sfft_status s;
  // the sparse part of the kernel-background block reads only R and the mask: it runs on the
  // plan's side stream, concurrently with the transforms, and is joined before the gather
  SFFT_CUDA_TRY(cudaEventRecord(p->evFork, st));
  SFFT_CUDA_TRY(cudaStreamWaitEvent(p->side, p->evFork, 0));
  { ProfScope ps(p, 9, p->side); s = sfft_launch_kb(p, R, mask, p->side, &nl); }
  if (s != SFFT_OK) return fail_joined(p, st, s);
  { ProfScope ps(p, 0, st); s = sfft_launch_row_fwd(p, R, reuseS ? nullptr : S, mask, true, p->T, p->pitchT, !p->fused, p->fused != 0, st, &nl); }
  if (s != SFFT_OK) return fail_joined(p, st, s);
  // the final moment reduction needs only the row pass: it follows the sparse chain on the side stream
  if (cudaEventRecord(p->evRow, st) != cudaSuccess || cudaStreamWaitEvent(p->side, p->evRow, 0) != cudaSuccess)
    return fail_joined(p, st, SFFT_ERR_CUDA);
  s = sfft_launch_moments(p, p->side, &nl);
  if (s != SFFT_OK) return fail_joined(p, st, s);
  if (cudaEventRecord(p->evJoin, p->side) != cudaSuccess) return fail_joined(p, st, SFFT_ERR_CUDA);
  if (p->fused) {
    // a2 (column pass, applies eta^q) + a3 (cross products + lag-pruned inverse along ky), fused
    ProfScope ps(p, 1, st);
    s = sfft_launch_colx(p, st, &nl);
  } else {
    { ProfScope ps(p, 1, st); s = sfft_launch_col_fwd(p, st, &nl); }
    if (s == SFFT_OK) s = sfft_launch_cross(p, st, &nl);
  }
  if (s != SFFT_OK) return fail_joined(p, st, s);
  SFFT_CUDA_TRY(cudaStreamWaitEvent(st, p->evJoin, 0));
  { ProfScope ps(p, 4, st); s = sfft_launch_lag_gather(p, A, b, st, &nl); }  // a3 (kx inverse on lag rows) + a4
  if (s != SFFT_OK) return s;
  p->launches[0] = nl;
  return SFFT_OK;
}

static bool build_args_ok(const sfft_plan* p, const double* R, const double* S, const unsigned char* mask,
                          const double* A, const double* b) {
  return p && R && S && A && b && aligned16(R) && aligned16(S) && aligned16(A) && aligned16(b) &&
         (!mask || aligned16(mask));
}

sfft_status sfft_build_system(sfft_plan* p, const double* R, const double* S, const unsigned char* mask,
                              double* A, double* b, void* stream) {
  if (!build_args_ok(p, R, S, mask, A, b)) return SFFT_ERR_INVALID_ARG;
  if (cuda_error_pending()) return SFFT_ERR_CUDA;
  return build_system_impl(p, R, S, mask, A, b, (cudaStream_t)stream);
}

sfft_status sfft_build_system_exact(sfft_plan* p, const double* R, const double* S, const unsigned char* mask,
                                    double* A, double* b, void* stream) {
  // every argument is validated before anything is enqueued
  if (!build_args_ok(p, R, S, mask, A, b)) return SFFT_ERR_INVALID_ARG;
  if (mask && !sfft_exact_supported(p->N, p->num_sms)) return SFFT_ERR_UNSUPPORTED;   // N > 2047 (some w > 5 models)
  if (cuda_error_pending()) return SFFT_ERR_CUDA;
  // the ordinary build on the unmasked images, then the masked pixels' rank-one terms are taken out
  sfft_status s = build_system_impl(p, R, S, nullptr, A, b, (cudaStream_t)stream);
  if (s != SFFT_OK || !mask) return s;
  int nl = p->launches[0];
  s = sfft_launch_exact_update(p, R, S, mask, A, b, (cudaStream_t)stream, &nl);
  if (s != SFFT_OK) return s;
  p->launches[0] = nl;
  return SFFT_OK;
}

sfft_status sfft_solve(sfft_plan* p, const double* A, const double* b, double* coeffs, int* info, void* stream) {
  if (!p || !A || !b || !coeffs) return SFFT_ERR_INVALID_ARG;
  if (cuda_error_pending()) return SFFT_ERR_CUDA;
  int nl = 0;
  sfft_status s;
  { ProfScope ps(p, 5, (cudaStream_t)stream); s = sfft_launch_solve(p, A, b, coeffs, info, (cudaStream_t)stream, &nl); }
  if (s != SFFT_OK) return s;
  p->launches[1] = nl;
  return SFFT_OK;
}

sfft_status sfft_subtract(sfft_plan* p, const double* R, const double* S, const double* coeffs, double* D,
                          void* stream) {
  if (!p || !R || !S || !coeffs || !D) return SFFT_ERR_INVALID_ARG;
  if (!aligned16(R) || !aligned16(S) || !aligned16(D) || D == R || D == S) return SFFT_ERR_INVALID_ARG;
  if (cuda_error_pending()) return SFFT_ERR_CUDA;
  int nl = (p->prepValid && p->prepR == R) ? p->launches[2] : 0;
  sfft_status s = sfft_launch_subtract(p, R, S, coeffs, D, (cudaStream_t)stream, &nl);
  if (s != SFFT_OK) return s;
  p->launches[2] = nl;
  return SFFT_OK;
}

// sfft_subtract_prepare without the argument checks (shared with the multi-template mode)
static sfft_status subtract_prepare_impl(sfft_plan* p, const double* R, cudaStream_t st) {
  int nl = 0;
  // ordered after everything already enqueued on `stream` (the build that used the scratch before),
  // then concurrent with whatever the caller enqueues next (typically sfft_solve)
  SFFT_CUDA_TRY(cudaEventRecord(p->evFork, st));
  SFFT_CUDA_TRY(cudaStreamWaitEvent(p->side, p->evFork, 0));
  sfft_status s = sfft_launch_subtract_rows(p, R, p->side, &nl);
  if (s != SFFT_OK) return fail_joined(p, st, s);
  if (cudaEventRecord(p->evPrep, p->side) != cudaSuccess) return fail_joined(p, st, SFFT_ERR_CUDA);
  p->prepR = R;
  p->prepValid = 1;
  p->launches[2] = nl;   // counted with the subtract call it belongs to
  return SFFT_OK;
}

sfft_status sfft_subtract_prepare(sfft_plan* p, const double* R, void* stream) {
  if (!p || !R || !aligned16(R)) return SFFT_ERR_INVALID_ARG;
  if (cuda_error_pending()) return SFFT_ERR_CUDA;
  return subtract_prepare_impl(p, R, (cudaStream_t)stream);
}

// One template of the multi-template mode on plan p and stream st: build (the science image's row transform
// and moments reused when reuseS), prepare, solve, subtract.  *nlTot receives the launches.
// after: the previous template's "build enqueued and finished" event when that template runs on another plan
// (the builds are throughput-bound, so they run one after the other and each solve falls beside the NEXT
// template's build instead of beside its peers' solves); p->evBuilt is recorded after this build.
static sfft_status mt_chain(sfft_plan* p, const double* Rk, const double* S, const unsigned char* mask, bool reuseS,
                            double* ck, int* infok, double* Dcur, cudaStream_t st, cudaEvent_t after, int* nlTot) {
  if (after) SFFT_CUDA_TRY(cudaStreamWaitEvent(st, after, 0));
  sfft_status s = build_system_impl(p, Rk, S, mask, p->mtA, p->mtB, st, reuseS);
  if (s != SFFT_OK) return s;
  SFFT_CUDA_TRY(cudaEventRecord(p->evBuilt, st));
  *nlTot += p->launches[0];
  // the coefficient-independent row transforms of the subtraction run beside the latency-bound solve
  s = subtract_prepare_impl(p, Rk, st);
  if (s != SFFT_OK) return s;
  int nl = 0;
  { ProfScope ps(p, 5, st); s = sfft_launch_solve(p, p->mtA, p->mtB, ck, infok, st, &nl); }
  if (s != SFFT_OK) return fail_joined(p, st, s);
  *nlTot += nl;
  nl = p->launches[2];
  s = sfft_launch_subtract(p, Rk, S, ck, Dcur, st, &nl);
  if (s != SFFT_OK) return s;
  *nlTot += nl;
  return SFFT_OK;
}

static bool mt_args_ok(const sfft_plan* p, const double* const* R, const double* S, const unsigned char* mask,
                       const double* scale, int n, const double* Dk, const double* coeffs, const double* out) {
  if (!p || !R || !S || !scale || !Dk || !coeffs || !out || n < 1 || n > SFFT_MAX_TEMPLATES) return false;
  if (!aligned16(S) || !aligned16(Dk) || !aligned16(out) || (mask && !aligned16(mask))) return false;
  const size_t npix = (size_t)p->H * p->W;
  for (int k = 0; k < n; ++k)
    if (!R[k] || !aligned16(R[k]) || R[k] == out || R[k] == S) return false;
  if (out == S || (out >= Dk && out < Dk + (size_t)n * npix)) return false;
  return true;
}

sfft_status sfft_multi_template_difference(sfft_plan* p, const double* const* R, const double* S,
                                           const unsigned char* mask, const double* scale, int n,
                                           double* Dk, double* coeffs, int* info, double* out, void* stream) {
  return sfft_multi_template_difference_plans(&p, 1, R, S, mask, scale, n, Dk, coeffs, info, out, stream);
}

sfft_status sfft_multi_template_difference_plans(sfft_plan* const* plans, int nplans, const double* const* R,
                                                 const double* S, const unsigned char* mask, const double* scale,
                                                 int n, double* Dk, double* coeffs, int* info, double* out,
                                                 void* stream) {
  if (!plans || nplans < 1 || nplans > SFFT_MAX_TEMPLATES || !plans[0]) return SFFT_ERR_INVALID_ARG;
  sfft_plan* p = plans[0];
  if (!mt_args_ok(p, R, S, mask, scale, n, Dk, coeffs, out)) return SFFT_ERR_INVALID_ARG;
  for (int q = 1; q < nplans; ++q) {
    const sfft_plan* h = plans[q];
    if (!h || h->H != p->H || h->W != p->W || h->w != p->w || h->DK != p->DK || h->DB != p->DB) return SFFT_ERR_INVALID_ARG;
    for (int r = 0; r < q; ++r)
      if (plans[r] == h) return SFFT_ERR_INVALID_ARG;
  }
  if (cuda_error_pending()) return SFFT_ERR_CUDA;
  cudaStream_t st = (cudaStream_t)stream;
  const size_t npix = (size_t)p->H * p->W;
  const int np = nplans < n ? nplans : n;
  // helper plans run their chains on their own work streams, forked from the caller stream here and joined
  // back into it before the median (and on every failure path): no host synchronisation
  if (np > 1) {
    SFFT_CUDA_TRY(cudaEventRecord(p->evWork, st));
    for (int q = 1; q < np; ++q) SFFT_CUDA_TRY(cudaStreamWaitEvent(plans[q]->work, p->evWork, 0));
  }
  auto join = [&]() {
    bool ok = true;
    for (int q = 1; q < np; ++q)
      ok = cudaEventRecord(plans[q]->evWork, plans[q]->work) == cudaSuccess &&
           cudaStreamWaitEvent(st, plans[q]->evWork, 0) == cudaSuccess && ok;
    if (!ok) cudaGetLastError();
    return ok;
  };
  const double* dptr[SFFT_MAX_TEMPLATES];
  int nlTot = 0;
  for (int k = 0; k < n; ++k) {
    sfft_plan* h = plans[k % np];
    double* Dcur = Dk + (size_t)k * npix;
    sfft_status s = mt_chain(h, R[k], S, mask, k >= np, coeffs + (size_t)k * p->N, info ? info + k : nullptr, Dcur,
                             k % np == 0 ? st : h->work, (np > 1 && k > 0) ? plans[(k - 1) % np]->evBuilt : nullptr, &nlTot);
    if (s != SFFT_OK) { join(); return s; }
    dptr[k] = Dcur;
  }
  if (!join()) return SFFT_ERR_CUDA;
  sfft_status s = sfft_median_combine(dptr, scale, n, npix, out, stream);
  if (s != SFFT_OK) return s;
  for (int q = 0; q < np; ++q) { plans[q]->launches[0] = 0; plans[q]->launches[1] = 0; plans[q]->launches[2] = 0; }
  p->launches[0] = nlTot + 1;   // the whole chain is reported as one "build" count of the first plan
  return SFFT_OK;
}

sfft_status sfft_probe_fp64(int kind, int iters, double* tflops, double* elapsed_ms, void* stream) {
  if (iters < 1 || kind < 0 || kind > 1) return SFFT_ERR_INVALID_ARG;
  double tf = 0, ms = 0;
  sfft_status s = sfft_run_probe(kind, iters, &tf, &ms, (cudaStream_t)stream);
  if (tflops) *tflops = tf;
  if (elapsed_ms) *elapsed_ms = ms;
  return s;
}

sfft_status sfft_profile_enable(sfft_plan* p, int on) {
  if (!p) return SFFT_ERR_INVALID_ARG;
  if (on && !p->prof_ev[0]) {
    for (int i = 0; i < 2 * SFFT_PROF_MAX; ++i)
      if (cudaEventCreate(&p->prof_ev[i]) != cudaSuccess) { cudaGetLastError(); return SFFT_ERR_CUDA; }
  }
  p->prof_on = on ? 1 : 0;
  return SFFT_OK;
}

sfft_status sfft_profile_read(sfft_plan* p, int stage, double* total_ms, int* count, int reset) {
  if (!p || stage < 0 || stage >= SFFT_NSTAGE) return SFFT_ERR_INVALID_ARG;
  // fold the pending event pairs into the per-stage totals (synchronises on those events)
  for (int i = 0; i < p->prof_n; ++i) {
    float ms = 0.f;
    if (cudaEventSynchronize(p->prof_ev[2 * i + 1]) != cudaSuccess ||
        cudaEventElapsedTime(&ms, p->prof_ev[2 * i], p->prof_ev[2 * i + 1]) != cudaSuccess) {
      cudaGetLastError();
      p->prof_n = 0;
      return SFFT_ERR_CUDA;
    }
    p->prof_ms[p->prof_stage[i]] += ms;
    p->prof_cnt[p->prof_stage[i]] += 1;
  }
  p->prof_n = 0;
  if (total_ms) *total_ms = p->prof_ms[stage];
  if (count) *count = p->prof_cnt[stage];
  if (reset) { p->prof_ms[stage] = 0.0; p->prof_cnt[stage] = 0; }
  return SFFT_OK;
}

int sfft_plan_fused(const sfft_plan* p) { return p ? p->fused : -1; }

sfft_status sfft_plan_set_solve_ctas(sfft_plan* p, int max_ctas) {
  if (!p || max_ctas < 0) return SFFT_ERR_INVALID_ARG;
  p->cholMaxCtas = max_ctas;
  return SFFT_OK;
}

int sfft_last_launch_count(const sfft_plan* p, int which) {
  if (!p || which < 0 || which > 2) return -1;
  return p->launches[which];
}

}  // extern "C"
