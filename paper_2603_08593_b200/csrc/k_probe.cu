// FP64 pipe probes: the measured "alu" roofline denominator.
//   kind 0: DFMA   -- 16 independent fused multiply-add chains per thread
//   kind 1: DMMA   -- mma.sync.aligned.m8n8k4 f64 (legacy tensor path; tcgen05 has no fp64 kind)
#include "sfft_common.cuh"

__global__ void __launch_bounds__(256) k_probe_dfma(int iters, double* sink) {
  double a[16];
  const double x = 1.0000001 + 1e-9 * threadIdx.x, y = 1e-9 * (blockIdx.x + 1);
#pragma unroll
  for (int i = 0; i < 16; ++i) a[i] = (double)i;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 16; ++i) a[i] = fma(a[i], x, y);
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < 16; ++i) s += a[i];
  if (s == 123.456) sink[0] = s;
}

__global__ void __launch_bounds__(256) k_probe_dmma(int iters, double* sink) {
  double c[8][2];
  const double a = 1.0 + 1e-9 * threadIdx.x, b = 1e-9 * (blockIdx.x + 1);
#pragma unroll
  for (int i = 0; i < 8; ++i) { c[i][0] = i; c[i][1] = -i; }
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 8; ++i)
      asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                   : "+d"(c[i][0]), "+d"(c[i][1])
                   : "d"(a), "d"(b));
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < 8; ++i) s += c[i][0] + c[i][1];
  if (s == 123.456) sink[0] = s;
}

sfft_status sfft_run_probe(int kind, int iters, double* tflops, double* ms, cudaStream_t st) {
  int dev = 0, sms = 0;
  SFFT_CUDA_TRY(cudaGetDevice(&dev));
  SFFT_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  double* sink = nullptr;
  SFFT_CUDA_TRY(cudaMalloc((void**)&sink, sizeof(double)));
  cudaEvent_t e0, e1;
  SFFT_CUDA_TRY(cudaEventCreate(&e0));
  SFFT_CUDA_TRY(cudaEventCreate(&e1));
  const int blocks = sms * 8, threads = 256;
  double flops = 0.0;
  for (int rep = 0; rep < 2; ++rep) {  // first repetition warms up
    SFFT_CUDA_TRY(cudaEventRecord(e0, st));
    if (kind == 0) {
      k_probe_dfma<<<blocks, threads, 0, st>>>(iters, sink);
      flops = (double)blocks * threads * (double)iters * 16.0 * 2.0;
    } else {
      k_probe_dmma<<<blocks, threads, 0, st>>>(iters, sink);
      flops = (double)blocks * (threads / 32) * (double)iters * 8.0 * (8.0 * 8.0 * 4.0 * 2.0);
    }
    SFFT_CUDA_TRY(cudaEventRecord(e1, st));
    SFFT_CUDA_TRY(cudaEventSynchronize(e1));
  }
  float t = 0.f;
  SFFT_CUDA_TRY(cudaEventElapsedTime(&t, e0, e1));
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(sink);
  *ms = t;
  *tflops = flops / ((double)t * 1e-3) / 1e12;
  return SFFT_OK;
}
