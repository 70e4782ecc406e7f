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
// Twiddles come from per-pass tables built on the host in long double (correctly rounded): the
// pass with radix R and sub-transform stride NS reads tab[(r-1)*NS + k] = exp(-2 pi i r k/(NS R)),
// so the lanes of a warp (consecutive k) read one contiguous segment per r through the
// read-only path; the inverse conjugates them.  The passes of one length are concatenated in
// pass order (fft_pass_table_size / fft_fill_pass_tables on the host, FftCfg<N>::tw_off on the
// device).
//
// The first pass can take its inputs straight from registers (fft_first_from_regs) and the last
// pass can leave its outputs in registers (fft_last_to_regs), so a kernel that loads from / stores
// to global memory in the butterfly's own access pattern never stages those elements in shared
// memory.
#pragma once
#include "sfft_common.cuh"

#ifndef SFFT_TW_TABLE
#define SFFT_TW_RECUR 1   // twiddles w^r, r >= 3, as products of w^1, w^2 (see fft_twiddle_load); -DSFFT_TW_TABLE: all from the table
#endif
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

// exp(-2 pi i m / 32), m in [0, 16): compile-time constants once m is (the rows' split/merge twiddles of
// one thread are w^(tr + e TPR) = w^tr * exp(-2 pi i e / (2 EPT)) -- one table load, EPT-1 constant products)
__host__ __device__ constexpr double sfft_cos32(int m) {
  constexpr double c[17] = {1.0, 0.98078528040323044913, 0.92387953251128675613, 0.83146961230254523708,
                            0.70710678118654752440, 0.55557023301960222474, 0.38268343236508977173,
                            0.19509032201612826785, 0.0, -0.19509032201612826785, -0.38268343236508977173,
                            -0.55557023301960222474, -0.70710678118654752440, -0.83146961230254523708,
                            -0.92387953251128675613, -0.98078528040323044913, -1.0};
  return c[m];
}
// a * exp(-2 pi i e / (2 EPT)),  e < EPT, EPT in {8, 16}
template <int EPT>
__device__ __forceinline__ cplx mul_split_root(cplx a, int e) {
  const int m = e * (16 / EPT);                     // exp(-2 pi i m/32) = cos(pi m/16) - i sin(pi m/16)
  const double cr = sfft_cos32(m), ci = -sfft_cos32(m < 8 ? 8 - m : m - 8) * (m < 8 ? 1.0 : 1.0);
  // sin(pi m/16) = cos(pi (8 - m)/16) for m <= 8 and = cos(pi (m - 8)/16) for m >= 8
  return cmake(fma(a.x, cr, -(a.y * ci)), fma(a.x, ci, a.y * cr));
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


// Radix plan per length (first radix = elements per thread).  Kept in one place for host and device.
__host__ __device__ constexpr int fft_num_passes(int N) {
  return (N == 8 || N == 16) ? 1 : (N <= 256 ? 2 : 3);
}
__host__ __device__ constexpr int fft_radix(int N, int pass) {
  switch (N) {
    case 8: return 8;
    case 16: return 16;
    case 32: return pass == 0 ? 8 : 4;
    case 64: return 8;
    case 128: return pass == 0 ? 16 : 8;
    case 256: return 16;
    case 512: return 8;
    case 1024: return pass == 0 ? 16 : 8;
    case 2048: return pass == 2 ? 8 : 16;
    case 4096: return 16;
    default: return 0;
  }
}
// stride NS of pass `pass` = product of the earlier radices
__host__ __device__ constexpr int fft_pass_ns(int N, int pass) {
  int ns = 1;
  for (int i = 0; i < pass; ++i) ns *= fft_radix(N, i);
  return ns;
}
// offset of a pass's twiddle block inside the concatenated table (pass 0 has none)
__host__ __device__ constexpr int fft_tw_off(int N, int pass) {
  int off = 0;
  for (int i = 1; i < pass; ++i) off += (fft_radix(N, i) - 1) * fft_pass_ns(N, i);
  return off;
}
__host__ __device__ constexpr int fft_pass_table_size(int N) {
  return fft_tw_off(N, fft_num_passes(N)) > 0 ? fft_tw_off(N, fft_num_passes(N)) : 1;
}

template <int N>
struct FftCfg {
  static constexpr int EPT = fft_radix(N, 0);   // first radix = elements per thread
  static constexpr int NPASS = fft_num_passes(N);
  static constexpr int PADSHIFT = (EPT == 8) ? 3 : 4;
  static constexpr int SEQ_STRIDE = N + (N >> PADSHIFT);
  static __host__ __device__ constexpr int phys(int n) { return n + (n >> PADSHIFT); }
};

// Butterfly m of thread tid -> (sequence, butterfly j).  SEQ_FAST: adjacent threads work on adjacent
// sequences (the column kernels, where adjacent sequences are adjacent in global memory).  Otherwise a
// sequence belongs to TPS = N/EPT consecutive threads in EVERY pass (butterflies j = t + m TPS of thread t), so
// the threads of one sequence exchange data only among themselves and may meet at a barrier of their own.
template <int NB, bool SEQ_FAST, int TPS>
__device__ __forceinline__ void fft_map(int tid, int m, int nth, int nseq, int& seq, int& j) {
  if (SEQ_FAST) { const int i = tid + m * nth; seq = i % nseq; j = i / nseq; }
  else { seq = tid / TPS; j = (tid - seq * TPS) + m * TPS; }
}

// twiddle + butterfly + Stockham store of one radix-R butterfly held in v[]
// a^2 and a*b for unit-modulus twiddles
__device__ __forceinline__ cplx csqr(cplx a) { return cmake(fma(a.x, a.x, -(a.y * a.y)), 2.0 * a.x * a.y); }
// The R-1 twiddles w^r, w = exp(-2 pi i k/(NS R)), of one butterfly.  SFFT_TW_RECUR: only w^1 (and w^2 for
// radix 16) come from the table; the others are products of at most three table values' powers
// (w^4 = (w^2)^2, w^8 = (w^4)^2, w^(a+b) = w^a w^b: depth <= 3 multiplications, error a few ulp), which
// trades ~13 table loads per radix-16 butterfly for ~50 fp64 operations: the row kernels are bound by
// the L1/shared-memory pipe with the fp64 pipe a third busy.
template <int N, int R, int NS>
__device__ __forceinline__ void fft_twiddle_load(cplx* t, int j, const cplx* __restrict__ tw) {
  if constexpr (NS > 1) {
    const int k = j & (NS - 1);
#ifdef SFFT_TW_RECUR
    t[1] = ldg2(tw + k);
    if constexpr (R >= 4) t[2] = ldg2(tw + NS + k);
#else
#pragma unroll
    for (int r = 1; r < R; ++r) t[r] = ldg2(tw + (r - 1) * NS + k);
#endif
  }
}
// completes t[] after the loads above have landed (no-op without SFFT_TW_RECUR)
template <int R, int NS>
__device__ __forceinline__ void fft_twiddle_complete(cplx* t) {
#ifdef SFFT_TW_RECUR
  if constexpr (NS > 1 && R >= 4) {
    t[3] = cmul(t[1], t[2]);
    if constexpr (R >= 8) {
      t[4] = csqr(t[2]);
      t[5] = cmul(t[1], t[4]);
      t[6] = cmul(t[2], t[4]);
      t[7] = cmul(t[3], t[4]);
    }
    if constexpr (R >= 16) {
      t[8] = csqr(t[4]);
#pragma unroll
      for (int r = 1; r < 8; ++r) t[8 + r] = cmul(t[r], t[8]);
    }
  }
#endif
}
template <int N, int R, int NS, int DIR>
__device__ __forceinline__ void fft_twiddle_apply(cplx* v, cplx* t) {
  if constexpr (NS > 1) {
    fft_twiddle_complete<R, NS>(t);
#pragma unroll
    for (int r = 1; r < R; ++r) {
      if (DIR > 0) t[r].y = -t[r].y;
      v[r] = cmul(v[r], t[r]);
    }
  }
  Dft<R, DIR>::run(v);
}
template <int N, int R, int NS, int DIR>
__device__ __forceinline__ void fft_twiddle_bfly(cplx* v, int j, const cplx* __restrict__ tw) {
  cplx t[R];
  fft_twiddle_load<N, R, NS>(t, j, tw);
  fft_twiddle_apply<N, R, NS, DIR>(v, t);
}
template <int N, int R, int NS>
__device__ __forceinline__ void fft_store(const cplx* v, cplx* base, int j) {
  using C = FftCfg<N>;
  const int k = j & (NS - 1);
  const int o = (j - k) * R + k;
#pragma unroll
  for (int r = 0; r < R; ++r) base[C::phys(o + r * NS)] = v[r];
}

// Barrier policies of the passes: the whole CTA (default), or a named barrier over the threads of one group of
// sequences (a kernel whose sequences are exchanged only inside such a group lets the groups drift apart).
struct FftSyncCta {
  __device__ __forceinline__ void operator()() const { __syncthreads(); }
};
template <int MAXID>
struct FftSyncNamed {
  int id, n;   // barrier 1..MAXID (immediate operands below, so the kernel reserves MAXID + 1 barriers, not 16); n threads, a multiple of 32
  __device__ __forceinline__ void operator()() const {
#define SFFT_BAR_CASE(I) case I: if constexpr (I <= MAXID) asm volatile("bar.sync " #I ", %0;\n" ::"r"(n) : "memory"); break;
    switch (id) {
      SFFT_BAR_CASE(1) SFFT_BAR_CASE(2) SFFT_BAR_CASE(3) SFFT_BAR_CASE(4)
      SFFT_BAR_CASE(5) SFFT_BAR_CASE(6) SFFT_BAR_CASE(7) SFFT_BAR_CASE(8)
      default: break;
    }
#undef SFFT_BAR_CASE
  }
};

// Pass 0 from registers: the calling thread supplies v[r] = x[seq][j + r*N/EPT], r < EPT, for the
// butterfly (seq, j) it chose (any one-to-one assignment of threads to butterflies).  Ends with a
// barrier unless the transform has a single pass and NOSYNC is set.
template <int N, int DIR, typename Sync = FftSyncCta>
__device__ __forceinline__ void fft_first_from_regs(cplx* v, cplx* s, int seq, int j, int seq_stride, Sync sync = Sync()) {
  using C = FftCfg<N>;
  Dft<C::EPT, DIR>::run(v);
  fft_store<N, C::EPT, 1>(v, s + seq * seq_stride, j);
  sync();
}

// One in-place pass shared memory -> shared memory.
template <int N, int R, int NS, int DIR, bool SEQ_FAST, typename Sync = FftSyncCta>
__device__ __forceinline__ void fft_pass(cplx* s, int tid, int nth, int nseq, const cplx* __restrict__ tw,
                                         const int seq_stride, Sync sync = Sync()) {
  using C = FftCfg<N>;
  constexpr int NB = N / R;        // butterflies per sequence
  constexpr int IT = C::EPT / R;   // butterflies per thread
  cplx v[IT][R], t[IT][R];
  // the twiddles do not depend on the data: their (global, L1/L2) loads are issued first so that
  // their latency hides under the shared-memory reads and the barrier
#pragma unroll
  for (int m = 0; m < IT; ++m) {
    int seq, j;
    fft_map<NB, SEQ_FAST, N / C::EPT>(tid, m, nth, nseq, seq, j);
    fft_twiddle_load<N, R, NS>(t[m], j, tw);
  }
#pragma unroll
  for (int m = 0; m < IT; ++m) {
    int seq, j;
    fft_map<NB, SEQ_FAST, N / C::EPT>(tid, m, nth, nseq, seq, j);
    const cplx* base = s + seq * seq_stride;
#pragma unroll
    for (int r = 0; r < R; ++r) v[m][r] = base[C::phys(j + r * NB)];
  }
  sync();
#pragma unroll
  for (int m = 0; m < IT; ++m) {
    int seq, j;
    fft_map<NB, SEQ_FAST, N / C::EPT>(tid, m, nth, nseq, seq, j);
    fft_twiddle_apply<N, R, NS, DIR>(v[m], t[m]);
    fft_store<N, R, NS>(v[m], s + seq * seq_stride, j);
  }
  sync();
}

// Last pass, outputs left in registers: butterfly m of the thread is (seq[m], j[m]) from fft_map
// and holds X[seq][j + r*N/R] in v[m*R + r].  No trailing barrier (nothing is written to smem).
template <int N, int R, int NS, int DIR, bool SEQ_FAST>
__device__ __forceinline__ void fft_pass_to_regs(const cplx* s, cplx* v, int tid, int nth, int nseq,
                                                 const cplx* __restrict__ tw, const int seq_stride) {
  using C = FftCfg<N>;
  constexpr int NB = N / R;
  constexpr int IT = C::EPT / R;
  cplx t[IT][R];
#pragma unroll
  for (int m = 0; m < IT; ++m) {
    int seq, j;
    fft_map<NB, SEQ_FAST, N / C::EPT>(tid, m, nth, nseq, seq, j);
    fft_twiddle_load<N, R, NS>(t[m], j, tw);
  }
#pragma unroll
  for (int m = 0; m < IT; ++m) {
    int seq, j;
    fft_map<NB, SEQ_FAST, N / C::EPT>(tid, m, nth, nseq, seq, j);
    const cplx* base = s + seq * seq_stride;
#pragma unroll
    for (int r = 0; r < R; ++r) v[m * R + r] = base[C::phys(j + r * NB)];
  }
#pragma unroll
  for (int m = 0; m < IT; ++m) fft_twiddle_apply<N, R, NS, DIR>(v + m * R, t[m]);
}

template <int N, int PASS, int DIR, bool SEQ_FAST, typename Sync = FftSyncCta>
__device__ __forceinline__ void fft_run_pass(cplx* s, int tid, int nth, int nseq, const cplx* __restrict__ tw,
                                             int seq_stride, Sync sync = Sync()) {
  fft_pass<N, fft_radix(N, PASS), fft_pass_ns(N, PASS), DIR, SEQ_FAST, Sync>(s, tid, nth, nseq,
                                                                             tw + fft_tw_off(N, PASS), seq_stride, sync);
}
template <int N, int PASS, int DIR, bool SEQ_FAST>
__device__ __forceinline__ void fft_run_pass_to_regs(const cplx* s, cplx* v, int tid, int nth, int nseq,
                                                     const cplx* __restrict__ tw, int seq_stride) {
  fft_pass_to_regs<N, fft_radix(N, PASS), fft_pass_ns(N, PASS), DIR, SEQ_FAST>(
      s, v, tid, nth, nseq, tw + fft_tw_off(N, PASS), seq_stride);
}

// Whole transform with the inputs in registers and the outputs left in shared memory
// (s[seq*seq_stride + phys(k)] = X[seq][k], visible to every thread on return).
// v[r] = x[seq][j + r*N/EPT] for the caller's butterfly (seq, j) = fft_map<N/EPT, SEQ_FAST>(tid).
// The CTA must have exactly nseq*N/EPT threads.  DIR = -1: X[k] = sum x[n] e^{-2 pi i nk/N};
// +1: e^{+...}; unnormalised.  A barrier must separate earlier readers of s from this call.
// Sync: the barrier between passes; a named barrier over one sequence's threads is valid when SEQ_FAST is
// false and a sequence's N/EPT threads are whole warps (they exchange data only among themselves); the
// caller then owes a CTA-wide barrier before threads of other sequences read s.
template <int N, int DIR, bool SEQ_FAST, typename Sync = FftSyncCta>
__device__ __forceinline__ void fft_regs_to_smem(cplx* v, cplx* s, int tid, int nth, int nseq,
                                                 const cplx* __restrict__ tw, int seq_stride, Sync sync = Sync()) {
  using C = FftCfg<N>;
  int seq, j;
  fft_map<N / C::EPT, SEQ_FAST, N / C::EPT>(tid, 0, nth, nseq, seq, j);
  fft_first_from_regs<N, DIR, Sync>(v, s, seq, j, seq_stride, sync);
  if constexpr (C::NPASS >= 2) fft_run_pass<N, 1, DIR, SEQ_FAST, Sync>(s, tid, nth, nseq, tw, seq_stride, sync);
  if constexpr (C::NPASS >= 3) fft_run_pass<N, 2, DIR, SEQ_FAST, Sync>(s, tid, nth, nseq, tw, seq_stride, sync);
}

// Whole transform registers -> registers.  On return, with RL = fft_radix(N, NPASS-1) and
// (seq_m, j_m) = fft_map<N/RL, SEQ_FAST>(tid + m*nth), v[m*RL + r] = X[seq_m][j_m + r*N/RL].
// No trailing barrier: a barrier must separate this call from the next writer of s.
template <int N, int DIR, bool SEQ_FAST>
__device__ __forceinline__ void fft_regs_to_regs(cplx* v, cplx* s, int tid, int nth, int nseq,
                                                 const cplx* __restrict__ tw, int seq_stride) {
  using C = FftCfg<N>;
  if constexpr (C::NPASS == 1) {
    Dft<C::EPT, DIR>::run(v);
  } else {
    int seq, j;
    fft_map<N / C::EPT, SEQ_FAST, N / C::EPT>(tid, 0, nth, nseq, seq, j);
    fft_first_from_regs<N, DIR>(v, s, seq, j, seq_stride);
    if constexpr (C::NPASS == 2) {
      fft_run_pass_to_regs<N, 1, DIR, SEQ_FAST>(s, v, tid, nth, nseq, tw, seq_stride);
    } else {
      fft_run_pass<N, 1, DIR, SEQ_FAST>(s, tid, nth, nseq, tw, seq_stride);
      fft_run_pass_to_regs<N, 2, DIR, SEQ_FAST>(s, v, tid, nth, nseq, tw, seq_stride);
    }
  }
}
