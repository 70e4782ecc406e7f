// The two steps that follow the differencing of one CCD:
//
//  k_median<N>      : multi-template combination, out = median_k(scale_k * D_k) per pixel
//                     (§2.3.2: the N_TEMP difference images are "normalized to a common
//                     photometric zero point ... and median-combined"; N_TEMP default 5).
//                     HBM-bound: N reads + 1 write of 8 bytes per pixel, 128-bit accesses, values
//                     sorted in registers by a fully unrolled insertion network.
//  k_aperture_flux  : Monte-Carlo limiting flux (§2.3.3: "aperture fluxes at 1024 randomly
//                     selected background positions ... deriving the 5 sigma threshold from their
//                     standard deviation"): one warp per position sums the hard-edged disc of pixels
//                     whose centres lie within `radius`; NaN if the disc leaves the frame or touches
//                     a masked pixel (readings L1, L2).  The positions are inputs.
//  k_aperture_stats : count, mean and population sigma of the kept fluxes, fixed-order tree sums.
//  k_cut_stamps     : three-channel (science, template, difference) stamps centred on candidate positions,
//                     the input of the real-bogus classifier (§2.3.4; NEXT-3).  A gather:
//                     one CTA per (candidate, channel), lanes along the stamp row; zero fill outside
//                     the frame, all-NaN stamp for a non-finite position (readings ST1-ST4).
//  k_resample<A>    : the step BEFORE the differencing (NEXT-4): Lanczos-A resampling of an image or a
//                     data-quality mask through an affine pixel map.
#include <math.h>
#include "sfft_common.cuh"

#define POST_MAXN SFFT_MAX_TEMPLATES

struct MedianParams {
  const double* D[POST_MAXN];
  double scale[POST_MAXN];
  double* out;
  size_t npix;
};

template <int N>
__device__ __forceinline__ double median_of(double* v) {
  // a NaN in any template makes the combined pixel NaN (reading M2; fmin/fmax below would
  // silently drop it)
  bool anynan = false;
#pragma unroll
  for (int i = 0; i < N; ++i) anynan |= (v[i] != v[i]);
  if (anynan) return nan("");
  // insertion sort with compile-time indices (stays in registers)
#pragma unroll
  for (int i = 1; i < N; ++i) {
#pragma unroll
    for (int j = i; j > 0; --j) {
      const double a = v[j - 1], b = v[j];
      v[j - 1] = fmin(a, b);
      v[j] = fmax(a, b);
    }
  }
  if (N & 1) return v[N / 2];
  return 0.5 * (v[(N - 1) / 2] + v[N / 2]);
}

template <int N>
__global__ void __launch_bounds__(256) k_median(MedianParams P) {
  const size_t npair = P.npix >> 1;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < npair; i += (size_t)gridDim.x * blockDim.x) {
    double a[N], b[N];
#pragma unroll
    for (int k = 0; k < N; ++k) {
      const double2 t = __ldcs(reinterpret_cast<const double2*>(P.D[k]) + i);
      a[k] = t.x * P.scale[k];
      b[k] = t.y * P.scale[k];
    }
    __stcs(reinterpret_cast<double2*>(P.out) + i, make_double2(median_of<N>(a), median_of<N>(b)));
  }
  if ((P.npix & 1) && blockIdx.x == 0 && threadIdx.x == 0) {   // odd tail
    double a[N];
#pragma unroll
    for (int k = 0; k < N; ++k) a[k] = P.D[k][P.npix - 1] * P.scale[k];
    P.out[P.npix - 1] = median_of<N>(a);
  }
}

template <int N>
static sfft_status launch_median_t(const MedianParams& P, cudaStream_t st) {
  size_t blocks = ((P.npix >> 1) + 255) / 256;
  const size_t cap = (size_t)sfft_device_sms() * 16;
  if (blocks > cap) blocks = cap;
  if (blocks < 1) blocks = 1;
  k_median<N><<<(unsigned)blocks, 256, 0, st>>>(P);
  SFFT_LAUNCH_CHECK();
  return SFFT_OK;
}

__global__ void __launch_bounds__(256) k_aperture_flux(const double* __restrict__ D, const unsigned char* __restrict__ mask,
                                                       int H, int W, const double* __restrict__ xs,
                                                       const double* __restrict__ ys, int n, double radius,
                                                       double* flux) {
  const int a = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), lane = threadIdx.x & 31;
  if (a >= n) return;
  const double x0 = xs[a], y0 = ys[a], r2 = radius * radius;
  const int ylo = (int)ceil(y0 - radius), yhi = (int)floor(y0 + radius);
  const int xlo = (int)ceil(x0 - radius), xhi = (int)floor(x0 + radius);
  // a non-finite position is dropped like one outside the frame (its int conversions are meaningless)
  const bool inside = isfinite(x0) && isfinite(y0) && ylo >= 0 && xlo >= 0 && yhi <= H - 1 && xhi <= W - 1;   // warp-uniform
  double acc = 0.0;
  int bad = 0;
  if (inside) {
    const int bw = xhi - xlo + 1, npx = bw * (yhi - ylo + 1);
    for (int e = lane; e < npx; e += 32) {
      const int y = ylo + e / bw, x = xlo + e % bw;
      const double dx = (double)x - x0, dy = (double)y - y0;
      if (dx * dx + dy * dy <= r2) {
        if (mask && mask[(size_t)y * W + x]) bad = 1;
        acc += D[(size_t)y * W + x];
      }
    }
  }
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) {
    acc += __shfl_xor_sync(0xffffffffu, acc, off);
    bad |= __shfl_xor_sync(0xffffffffu, bad, off);
  }
  if (lane == 0) flux[a] = (inside && !bad) ? acc : nan("");
}

// stats[0] = number of kept (non-NaN) fluxes, stats[1] = their mean, stats[2] = population sigma
__global__ void __launch_bounds__(1024) k_aperture_stats(const double* __restrict__ flux, int n, double* stats) {
  __shared__ double red[1024];
  __shared__ double s_mean;
  const int tid = threadIdx.x;
  auto block_sum = [&](double v) {
    red[tid] = v;
    __syncthreads();
    for (int off = 512; off > 0; off >>= 1) {
      if (tid < off) red[tid] += red[tid + off];
      __syncthreads();
    }
    const double r = red[0];
    __syncthreads();
    return r;
  };
  double cnt = 0.0, sum = 0.0;
  for (int i = tid; i < n; i += 1024) {
    const double f = flux[i];
    if (f == f) { cnt += 1.0; sum += f; }
  }
  const double N = block_sum(cnt), S = block_sum(sum);
  if (tid == 0) s_mean = N > 0.0 ? S / N : nan("");
  __syncthreads();
  const double mean = s_mean;
  double sq = 0.0;
  for (int i = tid; i < n; i += 1024) {
    const double f = flux[i];
    if (f == f) sq += (f - mean) * (f - mean);
  }
  const double Q = block_sum(sq);
  if (tid == 0) {
    stats[0] = N;
    stats[1] = mean;
    stats[2] = N > 0.0 ? sqrt(Q / N) : nan("");
  }
}

// ---- resampling onto another pixel grid --------------
// One thread per output pixel: affine map to the input frame, separable Lanczos-A weights
// L(t) = sinc(t) sinc(t/A) (exact zeros at the non-zero integers), normalised by their sum, 2A x 2A
// taps; outside the frame -> 0 and flagged.  MASK = true interpolates the 0/1 bad indicator and
// thresholds it (> thr -> 2, else 1; outside -> 2).
struct ResampleParams {
  const void* in;
  void* out;
  unsigned char* outside;   // nullable
  int Hin, Win, Hout, Wout;
  double M[6];
  double thr;
};

// The 2A Lanczos weights of one axis for the fractional offset f = x_in - floor(x_in) in [0, 1):
// tap k sits at t_k = f + (A - 1 - k).  sin(pi t_k) = (-1)^(A-1-k) sin(pi f) and
// sin(pi t_k / A) = sin(pi f / A) cos(pi m / A) + cos(pi f / A) sin(pi m / A), m = A - 1 - k, so one
// sinpi and one sincospi serve all taps; f = 0 gives exact zeros except the tap at t = 0.
__device__ __forceinline__ double rcp_fast(double a) {   // 1/a for normal a, ~1 ulp: seed + two fused Newton steps
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(a));
  const double e = fma(-a, r, 1.0);
  r = fma(r, fma(e, e, e), r);
  return fma(r, fma(-a, r, 1.0), r);
}

// cos(pi m / A) and sin(pi m / A) for A <= 4, |m| <= A, as compile-time constants
__host__ __device__ constexpr double lz_unit(int A, int num) {   // cos(pi num / A), num in [0, A]
  return num == 0 ? 1.0 : num == A ? -1.0 : 2 * num == A ? 0.0
       : A == 3 ? (num == 1 ? 0.5 : -0.5)
       : (num == 1 ? 0.70710678118654752440 : -0.70710678118654752440);   // A == 4, num = 1 or 3
}
__host__ __device__ constexpr double lz_cos(int A, int m) { return lz_unit(A, m < 0 ? -m : m); }
__host__ __device__ constexpr double lz_sin(int A, int m) {   // sin(x) = cos(pi/2 - x); here via the table
  const int am = m < 0 ? -m : m;
  const double v = am == 0 || am == A ? 0.0 : 2 * am == A ? 1.0
                 : A == 3 ? 0.86602540378443864676 : 0.70710678118654752440;
  return m < 0 ? -v : v;
}

template <int A>
__device__ __forceinline__ void lanczos_weights(double f, double* w) {
  const double s1 = sinpi(f);
  double sa, ca;
  sincospi(f / (double)A, &sa, &ca);
  const double pi2 = 9.86960440108935861883;   // pi^2
#pragma unroll
  for (int k = 0; k < 2 * A; ++k) {
    const int m = A - 1 - k;                    // t_k = f + m, m = A-1 .. -A
    const double t = f + (double)m;
    const double cm = lz_cos(A, m), sm = lz_sin(A, m);   // compile-time constants after unrolling
    const double sgn = (m & 1) ? -1.0 : 1.0;
    const double st = sgn * s1, sta = sa * cm + ca * sm;
    w[k] = (t == 0.0) ? 1.0 : (double)A * st * sta * rcp_fast(pi2 * t * t);
  }
}

template <int A, bool MASK>
__global__ void __launch_bounds__(256) k_resample(ResampleParams P) {
  const int xo = blockIdx.x * 32 + (threadIdx.x & 31), yo = blockIdx.y * 8 + (threadIdx.x >> 5);
  if (xo >= P.Wout || yo >= P.Hout) return;
  const double xi = P.M[0] + P.M[1] * (double)xo + P.M[2] * (double)yo;
  const double yi = P.M[3] + P.M[4] * (double)xo + P.M[5] * (double)yo;
  const double fx = floor(xi), fy = floor(yi);
  const size_t oidx = (size_t)yo * P.Wout + xo;
  const bool inside = fx - A + 1 >= 0.0 && fy - A + 1 >= 0.0 && fx + A <= (double)(P.Win - 1) && fy + A <= (double)(P.Hin - 1);
  if (!inside) {
    if (MASK) reinterpret_cast<unsigned char*>(P.out)[oidx] = 2;
    else reinterpret_cast<double*>(P.out)[oidx] = 0.0;
    if (P.outside) P.outside[oidx] = 1;
    return;
  }
  const int x0 = (int)fx - A + 1, y0 = (int)fy - A + 1;
  double wx[2 * A], wy[2 * A], sx = 0.0, sy = 0.0;
  lanczos_weights<A>(xi - fx, wx);
  lanczos_weights<A>(yi - fy, wy);
#pragma unroll
  for (int k = 0; k < 2 * A; ++k) {
    sx += wx[k];
    sy += wy[k];
  }
  double acc = 0.0;
#pragma unroll
  for (int j = 0; j < 2 * A; ++j) {
    double row = 0.0;
    const size_t base = (size_t)(y0 + j) * P.Win + x0;
#pragma unroll
    for (int k = 0; k < 2 * A; ++k) {
      const double v = MASK ? (reinterpret_cast<const unsigned char*>(P.in)[base + k] ? 1.0 : 0.0)
                            : reinterpret_cast<const double*>(P.in)[base + k];
      row += wx[k] * v;
    }
    acc += wy[j] * row;
  }
  const double val = acc / (sx * sy);
  if (MASK) reinterpret_cast<unsigned char*>(P.out)[oidx] = val > P.thr ? 2 : 1;
  else reinterpret_cast<double*>(P.out)[oidx] = val;
  if (P.outside) P.outside[oidx] = 0;
}

template <bool MASK>
static sfft_status launch_resample(const ResampleParams& P, int a, cudaStream_t st) {
  dim3 grid((P.Wout + 31) / 32, (P.Hout + 7) / 8);
  switch (a) {
    case 1: k_resample<1, MASK><<<grid, 256, 0, st>>>(P); break;
    case 2: k_resample<2, MASK><<<grid, 256, 0, st>>>(P); break;
    case 3: k_resample<3, MASK><<<grid, 256, 0, st>>>(P); break;
    case 4: k_resample<4, MASK><<<grid, 256, 0, st>>>(P); break;
    default: return SFFT_ERR_UNSUPPORTED;
  }
  SFFT_LAUNCH_CHECK();
  return SFFT_OK;
}


__global__ void __launch_bounds__(256) k_cut_stamps(const double* __restrict__ S, const double* __restrict__ R,
                                                    const double* __restrict__ D, int H, int W,
                                                    const double* __restrict__ xs, const double* __restrict__ ys,
                                                    int size, double* out) {
  const int k = blockIdx.x, ch = blockIdx.y;
  const double* img = ch == 0 ? S : (ch == 1 ? R : D);
  double* dst = out + ((size_t)k * 3 + ch) * size * size;
  const double x = xs[k], y = ys[k];
  const int npx = size * size;
  if (!(isfinite(x) && isfinite(y))) {
    for (int e = threadIdx.x; e < npx; e += blockDim.x) dst[e] = nan("");
    return;
  }
  // nearest pixel floor(x + 1/2); positions far outside the frame are clamped before the int
  // conversion (the stamp is all zero either way)
  const double lim = 1.0e9;
  const long long cx = (long long)floor(fmin(fmax(x, -lim), lim) + 0.5);
  const long long cy = (long long)floor(fmin(fmax(y, -lim), lim) + 0.5);
  const int half = size / 2;
  for (int e = threadIdx.x; e < npx; e += blockDim.x) {
    const int j = e / size, i = e - j * size;
    const long long yy = cy - half + j, xx = cx - half + i;
    dst[e] = (yy >= 0 && yy < H && xx >= 0 && xx < W) ? img[(size_t)yy * W + (size_t)xx] : 0.0;
  }
}

extern "C" {

sfft_status sfft_cut_stamps(const double* S, const double* R, const double* D, int H, int W, const double* xs,
                            const double* ys, int n, int size, double* out, void* stream) {
  if (!S || !R || !D || !xs || !ys || !out || H < 1 || W < 1 || n < 1 || size < 1 || size > 1024)
    return SFFT_ERR_INVALID_ARG;
  k_cut_stamps<<<dim3((unsigned)n, 3), 256, 0, (cudaStream_t)stream>>>(S, R, D, H, W, xs, ys, size, out);
  SFFT_LAUNCH_CHECK();
  return SFFT_OK;
}

sfft_status sfft_median_combine(const double* const* D, const double* scale, int n, size_t npix, double* out,
                                void* stream) {
  if (!D || !scale || !out || n < 1 || n > POST_MAXN || npix == 0) return SFFT_ERR_INVALID_ARG;
  MedianParams P;
  for (int k = 0; k < n; ++k) {
    if (!D[k] || (((uintptr_t)D[k]) & 15) || D[k] == out) return SFFT_ERR_INVALID_ARG;
    P.D[k] = D[k];
    P.scale[k] = scale[k];
  }
  if (((uintptr_t)out) & 15) return SFFT_ERR_INVALID_ARG;
  P.out = out; P.npix = npix;
  cudaStream_t st = (cudaStream_t)stream;
  switch (n) {
    case 1: return launch_median_t<1>(P, st);
    case 2: return launch_median_t<2>(P, st);
    case 3: return launch_median_t<3>(P, st);
    case 4: return launch_median_t<4>(P, st);
    case 5: return launch_median_t<5>(P, st);
    case 6: return launch_median_t<6>(P, st);
    case 7: return launch_median_t<7>(P, st);
    case 8: return launch_median_t<8>(P, st);
    default: return launch_median_t<9>(P, st);
  }
}

sfft_status sfft_aperture_stats(const double* D, const unsigned char* mask, int H, int W, const double* xs,
                                const double* ys, int n, double radius, double* flux, double* stats,
                                void* stream) {
  if (!D || !xs || !ys || !flux || !stats || H < 1 || W < 1 || n < 1 || !(radius > 0.0) || radius > 64.0)
    return SFFT_ERR_INVALID_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  k_aperture_flux<<<(n + 7) / 8, 256, 0, st>>>(D, mask, H, W, xs, ys, n, radius, flux);
  SFFT_LAUNCH_CHECK();
  k_aperture_stats<<<1, 1024, 0, st>>>(flux, n, stats);
  SFFT_LAUNCH_CHECK();
  return SFFT_OK;
}

sfft_status sfft_resample_affine(const double* in, int Hin, int Win, const double* M, int a, double* out,
                                 int Hout, int Wout, unsigned char* outside, void* stream) {
  if (!in || !M || !out || Hin < 1 || Win < 1 || Hout < 1 || Wout < 1 || in == out) return SFFT_ERR_INVALID_ARG;
  ResampleParams P;
  P.in = in; P.out = out; P.outside = outside; P.Hin = Hin; P.Win = Win; P.Hout = Hout; P.Wout = Wout; P.thr = 0.0;
  for (int i = 0; i < 6; ++i) P.M[i] = M[i];
  return launch_resample<false>(P, a, (cudaStream_t)stream);
}

sfft_status sfft_resample_mask_affine(const unsigned char* in, int Hin, int Win, const double* M, int a,
                                      double threshold, unsigned char* out, int Hout, int Wout, void* stream) {
  if (!in || !M || !out || Hin < 1 || Win < 1 || Hout < 1 || Wout < 1 || in == out) return SFFT_ERR_INVALID_ARG;
  ResampleParams P;
  P.in = in; P.out = out; P.outside = nullptr; P.Hin = Hin; P.Win = Win; P.Hout = Hout; P.Wout = Wout;
  P.thr = threshold;
  for (int i = 0; i < 6; ++i) P.M[i] = M[i];
  return launch_resample<true>(P, a, (cudaStream_t)stream);
}

}  // extern "C"
