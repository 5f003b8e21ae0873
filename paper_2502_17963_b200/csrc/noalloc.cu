// noalloc.cu — the one entry point of the library that allocates nothing: bqc_sum_fixed_noalloc.
//
// Some callers cannot call cudaMalloc: code under CUDA-graph capture, tight serving loops, harnesses that forbid it.
// This is a two-stage variant of the fixed-order final sum of the (T) path (final_sum_kernel, SURVEY.md §8(a) row
// a5: E(T) = sum of e_ijk in a fixed order, no floating-point atomics).  The single-block kernel of the main path
// walks the whole array with 1024 threads; here stage 1 lets one CTA per 4096-element chunk write its partial sum
// into SCRATCH, and stage 2 sums the partials with one CTA.  The scratch is the file-scope array below — device
// memory that every GPU that loads libbqc_t.so holds until the process exits (32 KiB) — so the call performs no
// cudaMalloc / cudaFree / cudaMallocAsync and no allocating library routine.
//
// * The array's name is a host-side stand-in in host code, not a device address: its address is looked up once per
//   device, with that device current, by cudaGetSymbolAddress, and that pointer is what the kernels receive.
// * Every call on a device shares the array and finds the last call's contents in it.  Nothing has to start at
//   zero: stage 1 writes every slot stage 2 reads (slots [0, ceil(n / 4096))), and slots beyond are never read.
// * Calls that overlap on the GPU (two streams, or two host threads on one device) RACE on the array; order them
//   on one stream or with events.
#include "kernels.cuh"

namespace bqc {

namespace {

constexpr int kNaChunk = 4096;          // elements per stage-1 CTA
constexpr int kNaMaxPartials = 4096;    // scratch slots: n <= kNaChunk * kNaMaxPartials = 16 777 216 elements
constexpr int kNaThreads = 256;

static __device__ __align__(256) double g_noalloc_scratch[kNaMaxPartials];   // 32 KiB per GPU, held until exit

// scratch[b] = sum of x[b*4096 .. min(n, (b+1)*4096)) — thread t adds elements t, t+256, ... in order, then a fixed
// shared-memory tree: the result depends on n and the data only.
__global__ void __launch_bounds__(kNaThreads) noalloc_partial_kernel(const double* __restrict__ x, long long n,
                                                                     double* __restrict__ scratch) {
  __shared__ double red[kNaThreads];
  const long long lo = (long long)blockIdx.x * kNaChunk;
  const long long hi = lo + kNaChunk < n ? lo + kNaChunk : n;
  double s = 0.0;
  for (long long i = lo + threadIdx.x; i < hi; i += kNaThreads) s += x[i];
  red[threadIdx.x] = s;
  __syncthreads();
  for (int off = kNaThreads / 2; off > 0; off >>= 1) {
    if (threadIdx.x < off) red[threadIdx.x] += red[threadIdx.x + off];
    __syncthreads();
  }
  if (threadIdx.x == 0) scratch[blockIdx.x] = red[0];
}

// *out = sum of scratch[0 .. m) in a fixed order (one CTA); m = 0 gives 0.
__global__ void __launch_bounds__(kNaThreads) noalloc_final_kernel(const double* __restrict__ scratch, int m,
                                                                   double* __restrict__ out) {
  __shared__ double red[kNaThreads];
  double s = 0.0;
  for (int i = threadIdx.x; i < m; i += kNaThreads) s += scratch[i];
  red[threadIdx.x] = s;
  __syncthreads();
  for (int off = kNaThreads / 2; off > 0; off >>= 1) {
    if (threadIdx.x < off) red[threadIdx.x] += red[threadIdx.x + off];
    __syncthreads();
  }
  if (threadIdx.x == 0) *out = red[0];
}

// Device address of the scratch array on the current device: cudaGetSymbolAddress once per device.
int scratch_address(double** out) {
  static double* addr[64] = {};
  int dev = 0;
  BQC_CUDA_OK(cudaGetDevice(&dev));
  if (dev < 0 || dev >= 64) {
    set_error(BQC_ERR_DEVICE, "bqc_sum_fixed_noalloc: device ordinal %d outside [0, 64)", dev);
    return BQC_ERR_DEVICE;
  }
  if (!addr[dev]) {
    double* p = nullptr;
    BQC_CUDA_OK(cudaGetSymbolAddress(reinterpret_cast<void**>(&p), g_noalloc_scratch));
    if (!p) {
      set_error(BQC_ERR_CUDA, "bqc_sum_fixed_noalloc: cudaGetSymbolAddress returned a null address");
      return BQC_ERR_CUDA;
    }
    addr[dev] = p;
  }
  *out = addr[dev];
  return BQC_OK;
}

}  // namespace
}  // namespace bqc

using namespace bqc;

extern "C" {

size_t bqc_sum_fixed_noalloc_max(void) { return (size_t)kNaChunk * kNaMaxPartials; }

int bqc_sum_fixed_noalloc(const double* x_dev, size_t n, double* out_dev, void* stream_v) {
  clear_error();
  cudaStream_t stream = static_cast<cudaStream_t>(stream_v);
  if (n > bqc_sum_fixed_noalloc_max()) {
    set_error(BQC_ERR_INVALID_SIZE,
              "bqc_sum_fixed_noalloc: n = %zu exceeds the maximum of %zu elements the static scratch array covers "
              "(%d partial sums of %d elements); use bqc_sum_in_order or split the array",
              n, bqc_sum_fixed_noalloc_max(), kNaMaxPartials, kNaChunk);
    return BQC_ERR_INVALID_SIZE;
  }
  BQC_TRY(check_device());
  BQC_TRY(check_device_ptr(out_dev, "out_dev"));
  if (n > 0) BQC_TRY(check_device_ptr(x_dev, "x_dev"));
  double* scratch = nullptr;
  BQC_TRY(scratch_address(&scratch));
  const int m = (int)((n + kNaChunk - 1) / kNaChunk);
  if (m > 0) {
    noalloc_partial_kernel<<<m, kNaThreads, 0, stream>>>(x_dev, (long long)n, scratch);
    count_launch();
    BQC_CUDA_OK(cudaGetLastError());
  }
  noalloc_final_kernel<<<1, kNaThreads, 0, stream>>>(scratch, m, out_dev);
  count_launch();
  BQC_CUDA_OK(cudaGetLastError());
  return BQC_OK;
}

}  // extern "C"
