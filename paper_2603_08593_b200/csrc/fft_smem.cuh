// Block-cooperative fp64 complex FFT in shared memory (Stockham radix-16/8/4 passes).
//
// Used by the forward row pass (length W/2, real rows packed as complex), the forward column
// pass (length H) and the inverse row pass of sfft_subtract (north_star subsystem (2): "batched
// fp64 2D R2C/C2R FFTs with shared-memory staged radix passes").
//
// Layout: a CTA owns `nseq` sequences of length N; sequence q lives at s[q*SEQ_STRIDE + phys(n)],
// phys(n) = n + (n >> PADSHIFT): one 16-byte pad per first-radix group, which makes the
// stride-R stores of the first pass bank-conflict free while contiguous accesses stay contiguous
// inside every aligned 8-lane phase.  The CTA has exactly nseq*N/EPT threads; each thread holds
// EPT complex values in registers per pass, so every pass is: load all -> barrier -> twiddle +
// register butterfly -> store all -> barrier (in place, no ping-pong buffer).
//
// Twiddles come from a table tw[m] = exp(-2 pi i m / N) built on the host in long double
// (correctly rounded), read through the read-only path; the inverse conjugates them.
#pragma once
#include "sfft_common.cuh"

#define SFFT_SQRT1_2 0.70710678118654752440
#define SFFT_COS_PI_8 0.92387953251128675613
#define SFFT_SIN_PI_8 0.38268343236508977173

template <int DIR>
__device__ __forceinline__ cplx mul_qi(cplx a) {  // a * exp(DIR * i pi/2)
  return DIR > 0 ? cmul_pi(a) : cmul_mi(a);
}
template <int DIR>
__device__ __forceinline__ cplx mul_w8_1(cplx a) {  // a * exp(DIR * 2 pi i /8)
  return cmake(SFFT_SQRT1_2 * (a.x - DIR * a.y), SFFT_SQRT1_2 * (a.y + DIR * a.x));
}
template <int DIR>
__device__ __forceinline__ cplx mul_w8_3(cplx a) {  // a * exp(DIR * 2 pi i 3/8)
  return cmake(SFFT_SQRT1_2 * (-a.x - DIR * a.y), SFFT_SQRT1_2 * (DIR * a.x - a.y));
}
template <int DIR>
__device__ __forceinline__ cplx mul_const(cplx a, double cr, double ci) {  // a * (cr + i DIR ci)
  return cmake(fma(a.x, cr, -(DIR * ci) * a.y), fma(a.x, DIR * ci, a.y * cr));
}
// a * exp(DIR * 2 pi i M / 16), M in [0, 9]
template <int M, int DIR>
__device__ __forceinline__ cplx mul_w16(cplx a) {
  if constexpr (M == 0) return a;
  else if constexpr (M == 1) return mul_const<DIR>(a, SFFT_COS_PI_8, SFFT_SIN_PI_8);
  else if constexpr (M == 2) return mul_w8_1<DIR>(a);
  else if constexpr (M == 3) return mul_const<DIR>(a, SFFT_SIN_PI_8, SFFT_COS_PI_8);
  else if constexpr (M == 4) return mul_qi<DIR>(a);
  else if constexpr (M == 6) return mul_w8_3<DIR>(a);
  else if constexpr (M == 9) return mul_const<DIR>(a, -SFFT_COS_PI_8, -SFFT_SIN_PI_8);
  else return a;
}

template <int DIR>
__device__ __forceinline__ void dft4(cplx& x0, cplx& x1, cplx& x2, cplx& x3) {
  cplx a = cadd(x0, x2), b = csub(x0, x2), c = cadd(x1, x3), d = mul_qi<DIR>(csub(x1, x3));
  x0 = cadd(a, c);
  x1 = cadd(b, d);
  x2 = csub(a, c);
  x3 = csub(b, d);
}

template <int R, int DIR>
struct Dft;

template <int DIR>
struct Dft<2, DIR> {
  static __device__ __forceinline__ void run(cplx* v) {
    cplx t = v[0];
    v[0] = cadd(t, v[1]);
    v[1] = csub(t, v[1]);
  }
};
template <int DIR>
struct Dft<4, DIR> {
  static __device__ __forceinline__ void run(cplx* v) { dft4<DIR>(v[0], v[1], v[2], v[3]); }
};
template <int DIR>
struct Dft<8, DIR> {
  // n = n1 + 2 n2, k = 4 k1 + k2:  X[4k1+k2] = T0[k2] + (-1)^k1 w8^k2 T1[k2]
  static __device__ __forceinline__ void run(cplx* v) {
    dft4<DIR>(v[0], v[2], v[4], v[6]);
    dft4<DIR>(v[1], v[3], v[5], v[7]);
    cplx t1 = mul_w8_1<DIR>(v[3]);
    cplx t2 = mul_qi<DIR>(v[5]);
    cplx t3 = mul_w8_3<DIR>(v[7]);
    cplx e0 = v[0], e1 = v[2], e2 = v[4], e3 = v[6], o0 = v[1];
    v[0] = cadd(e0, o0);
    v[4] = csub(e0, o0);
    v[1] = cadd(e1, t1);
    v[5] = csub(e1, t1);
    v[2] = cadd(e2, t2);
    v[6] = csub(e2, t2);
    v[3] = cadd(e3, t3);
    v[7] = csub(e3, t3);
  }
};
template <int DIR>
struct Dft<16, DIR> {
  // n = n1 + 4 n2, k = 4 k1 + k2:  X[4k1+k2] = sum_n1 w4^(n1 k1) w16^(n1 k2) T_n1[k2]
  static __device__ __forceinline__ void run(cplx* v) {
    dft4<DIR>(v[0], v[4], v[8], v[12]);   // T0[k2] at v[4 k2]
    dft4<DIR>(v[1], v[5], v[9], v[13]);   // T1[k2] at v[1 + 4 k2]
    dft4<DIR>(v[2], v[6], v[10], v[14]);  // T2
    dft4<DIR>(v[3], v[7], v[11], v[15]);  // T3
    // twiddle T_n1[k2] by w16^(n1 k2)
    v[5] = mul_w16<1, DIR>(v[5]);
    v[9] = mul_w16<2, DIR>(v[9]);
    v[13] = mul_w16<3, DIR>(v[13]);
    v[6] = mul_w16<2, DIR>(v[6]);
    v[10] = mul_w16<4, DIR>(v[10]);
    v[14] = mul_w16<6, DIR>(v[14]);
    v[7] = mul_w16<3, DIR>(v[7]);
    v[11] = mul_w16<6, DIR>(v[11]);
    v[15] = mul_w16<9, DIR>(v[15]);
    // DFT4 over n1 for each k2: inputs v[4 k2 + n1] -> outputs X[4 k1 + k2]
    dft4<DIR>(v[0], v[1], v[2], v[3]);      // k2 = 0 -> X[0], X[4], X[8], X[12] at v[0..3]
    dft4<DIR>(v[4], v[5], v[6], v[7]);      // k2 = 1 -> X[1], X[5], X[9], X[13] at v[4..7]
    dft4<DIR>(v[8], v[9], v[10], v[11]);    // k2 = 2
    dft4<DIR>(v[12], v[13], v[14], v[15]);  // k2 = 3
    // now v[4 k2 + k1] = X[4 k1 + k2]: transpose the 4x4 register tile to natural order
    cplx t;
#define SFFT_SWAP(i, j) t = v[i]; v[i] = v[j]; v[j] = t;
    SFFT_SWAP(1, 4) SFFT_SWAP(2, 8) SFFT_SWAP(3, 12) SFFT_SWAP(6, 9) SFFT_SWAP(7, 13) SFFT_SWAP(11, 14)
#undef SFFT_SWAP
  }
};

template <int N>
struct FftCfg {
  // first radix = elements per thread
  static constexpr int EPT = (N == 8 || N == 32 || N == 64 || N == 512) ? 8 : 16;
  static constexpr int PADSHIFT = (EPT == 8) ? 3 : 4;
  static constexpr int SEQ_STRIDE = N + (N >> PADSHIFT);
  static __host__ __device__ constexpr int phys(int n) { return n + (n >> PADSHIFT); }
};

template <int N, int R, int NS, int DIR>
__device__ __forceinline__ void fft_pass(cplx* s, int tid, int nth, const cplx* __restrict__ tw,
                                         const int seq_stride) {
  using C = FftCfg<N>;
  constexpr int NB = N / R;        // butterflies per sequence
  constexpr int IT = C::EPT / R;   // butterflies per thread
  cplx v[IT][R];
#pragma unroll
  for (int m = 0; m < IT; ++m) {
    const int i = tid + m * nth;
    const int seq = i / NB, j = i & (NB - 1);
    const cplx* base = s + seq * seq_stride;
#pragma unroll
    for (int r = 0; r < R; ++r) v[m][r] = base[C::phys(j + r * NB)];
  }
  __syncthreads();
#pragma unroll
  for (int m = 0; m < IT; ++m) {
    const int i = tid + m * nth;
    const int seq = i / NB, j = i & (NB - 1);
    const int k = j & (NS - 1);
    if constexpr (NS > 1) {
#pragma unroll
      for (int r = 1; r < R; ++r) {
        cplx t = ldg2(tw + r * k * (N / (NS * R)));
        if (DIR > 0) t.y = -t.y;
        v[m][r] = cmul(v[m][r], t);
      }
    }
    Dft<R, DIR>::run(v[m]);
    cplx* base = s + seq * seq_stride;
    const int o = (j - k) * R + k;
#pragma unroll
    for (int r = 0; r < R; ++r) base[C::phys(o + r * NS)] = v[m][r];
  }
  __syncthreads();
}

// In-place FFT of every sequence the CTA holds.  All nth = nseq*N/EPT threads must call it.
// On entry the data must be visible (a __syncthreads after the producer's stores); on exit the
// results are visible to every thread.  DIR = -1: X[k] = sum x[n] e^{-2 pi i nk/N}; +1: e^{+...},
// unnormalised.
template <int N, int DIR>
__device__ __forceinline__ void fft_smem(cplx* s, int tid, int nth, const cplx* __restrict__ tw,
                                         const int seq_stride = FftCfg<N>::SEQ_STRIDE) {
  if constexpr (N == 8) {
    fft_pass<N, 8, 1, DIR>(s, tid, nth, tw, seq_stride);
  } else if constexpr (N == 16) {
    fft_pass<N, 16, 1, DIR>(s, tid, nth, tw, seq_stride);
  } else if constexpr (N == 32) {
    fft_pass<N, 8, 1, DIR>(s, tid, nth, tw, seq_stride);
    fft_pass<N, 4, 8, DIR>(s, tid, nth, tw, seq_stride);
  } else if constexpr (N == 64) {
    fft_pass<N, 8, 1, DIR>(s, tid, nth, tw, seq_stride);
    fft_pass<N, 8, 8, DIR>(s, tid, nth, tw, seq_stride);
  } else if constexpr (N == 128) {
    fft_pass<N, 16, 1, DIR>(s, tid, nth, tw, seq_stride);
    fft_pass<N, 8, 16, DIR>(s, tid, nth, tw, seq_stride);
  } else if constexpr (N == 256) {
    fft_pass<N, 16, 1, DIR>(s, tid, nth, tw, seq_stride);
    fft_pass<N, 16, 16, DIR>(s, tid, nth, tw, seq_stride);
  } else if constexpr (N == 512) {
    fft_pass<N, 8, 1, DIR>(s, tid, nth, tw, seq_stride);
    fft_pass<N, 8, 8, DIR>(s, tid, nth, tw, seq_stride);
    fft_pass<N, 8, 64, DIR>(s, tid, nth, tw, seq_stride);
  } else if constexpr (N == 1024) {
    fft_pass<N, 16, 1, DIR>(s, tid, nth, tw, seq_stride);
    fft_pass<N, 8, 16, DIR>(s, tid, nth, tw, seq_stride);
    fft_pass<N, 8, 128, DIR>(s, tid, nth, tw, seq_stride);
  } else if constexpr (N == 2048) {
    fft_pass<N, 16, 1, DIR>(s, tid, nth, tw, seq_stride);
    fft_pass<N, 16, 16, DIR>(s, tid, nth, tw, seq_stride);
    fft_pass<N, 8, 256, DIR>(s, tid, nth, tw, seq_stride);
  } else if constexpr (N == 4096) {
    fft_pass<N, 16, 1, DIR>(s, tid, nth, tw, seq_stride);
    fft_pass<N, 16, 16, DIR>(s, tid, nth, tw, seq_stride);
    fft_pass<N, 16, 256, DIR>(s, tid, nth, tw, seq_stride);
  } else {
    static_assert(N == 8, "unsupported FFT length");
  }
}
