// peak.cu — register-resident FP64 peak microbenchmarks: the denominator of the
// headline "% of FP64 tensor-core peak" is MEASURED in the same run, not taken from a datasheet.
#include "kernels.cuh"

namespace bqc {

namespace {
constexpr int kChains = 16;

template <int KIND>
__global__ void __launch_bounds__(256) fp64_peak_kernel(int iters, double seed, double* sink) {
  // KIND 0: DMMA only, 1: DFMA only, 2: both interleaved in the same warp
  double c0[kChains], c1[kChains], f[kChains];
  const double a = seed + threadIdx.x * 1e-9, b = 1.0 - seed;
#pragma unroll
  for (int n = 0; n < kChains; ++n) { c0[n] = n; c1[n] = -n; f[n] = n * 0.5; }
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int n = 0; n < kChains; ++n) {
      if (KIND == 0 || KIND == 2) dmma_884(c0[n], c1[n], a, b);
      if (KIND == 1 || KIND == 2) f[n] = fma(f[n], a, b);
    }
  }
  double s = 0.0;
#pragma unroll
  for (int n = 0; n < kChains; ++n) s += c0[n] + c1[n] + f[n];
  if (s == 123.456) sink[0] = s;   // keep the work alive
}

template <int KIND>
double run_kind(double seconds, cudaStream_t s) {
  const int sms = 148 * 1;
  int dev = 0, nsm = sms;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
  const int grid = nsm * 4, block = 256;   // 32 warps per SM, 8 per scheduler
  double* sink = nullptr;
  if (cudaMalloc(&sink, 8) != cudaSuccess) return -1.0;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  const int iters = 20000;
  // flops per launch
  const double warps = (double)grid * block / 32.0;
  double flops_per_launch = 0.0;
  if (KIND == 0 || KIND == 2) flops_per_launch += warps * iters * kChains * 512.0;          // 8x8x4 MMA = 256 FMA
  if (KIND == 1 || KIND == 2) flops_per_launch += warps * iters * kChains * 32.0 * 2.0;
  fp64_peak_kernel<KIND><<<grid, block, 0, s>>>(iters, 0.25, sink);   // warm-up
  cudaStreamSynchronize(s);
  double total_ms = 0.0, total_flops = 0.0;
  while (total_ms < seconds * 1e3) {
    cudaEventRecord(e0, s);
    for (int rep = 0; rep < 4; ++rep) fp64_peak_kernel<KIND><<<grid, block, 0, s>>>(iters, 0.25, sink);
    cudaEventRecord(e1, s);
    if (cudaEventSynchronize(e1) != cudaSuccess) { total_ms = -1; break; }
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    total_ms += ms;
    total_flops += 4 * flops_per_launch;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(sink);
  if (total_ms <= 0) return -1.0;
  return total_flops / (total_ms * 1e-3) * 1e-12;
}
}  // namespace

double run_fp64_peak(int kind, double seconds, cudaStream_t s) {
  switch (kind) {
    case 0: return run_kind<0>(seconds, s);
    case 1: return run_kind<1>(seconds, s);
    case 2: return run_kind<2>(seconds, s);
  }
  return -1.0;
}

}  // namespace bqc
