// gemm_nt.cu — host side of the tile-GEMM engine: tensor-map encoding and launch.
#include "gemm_nt.cuh"

#include <mutex>

namespace bqc {

typedef CUresult (*PFN_encodeTiled)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*,
                                    const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                    const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                    CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static PFN_encodeTiled get_encode_fn() {
  static PFN_encodeTiled fn = nullptr;
  static std::once_flag once;
  std::call_once(once, [] {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    // the driver entry point is resolved at run time so that libbqc_t.so does not link libcuda
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<PFN_encodeTiled>(p);
  });
  return fn;
}

int make_tensor_map_f64(CUtensorMap* out, const void* base, const unsigned long long dims[4],
                        const unsigned long long strides_bytes[4], unsigned box1, unsigned box2) {
  PFN_encodeTiled enc = get_encode_fn();
  if (!enc) {
    set_error(BQC_ERR_CUDA, "cuTensorMapEncodeTiled entry point not available");
    return BQC_ERR_CUDA;
  }
  cuuint64_t gdim[4] = {dims[0], dims[1], dims[2], dims[3]};
  cuuint64_t gstr[3] = {strides_bytes[1], strides_bytes[2], strides_bytes[3]};
  cuuint32_t box[4] = {(cuuint32_t)kBK, box1, box2, 1};
  cuuint32_t estr[4] = {1, 1, 1, 1};
  CUresult r = enc(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, const_cast<void*>(base), gdim, gstr, box,
                   estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                   CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    set_error(BQC_ERR_CUDA,
              "cuTensorMapEncodeTiled failed (%d): dims %llu %llu %llu %llu strides %llu %llu %llu box %u %u",
              (int)r, dims[0], dims[1], dims[2], dims[3], strides_bytes[1], strides_bytes[2],
              strides_bytes[3], box1, box2);
    return BQC_ERR_CUDA;
  }
  return BQC_OK;
}

int device_sm_count() {
  // per device: a process may drive several GPUs (cudaSetDevice) through the same library
  static int sms[64] = {};
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return 0;
  if (dev < 0 || dev >= 64) {
    int n = 0;
    return cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess ? n : 0;
  }
  if (sms[dev] == 0 && cudaDeviceGetAttribute(&sms[dev], cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
    return 0;
  return sms[dev];
}

// Modelled relative time of an N extent covered by tiles of 8*nf columns: padded columns times a per-tile
// efficiency factor (measured: the tensor pipe is ~0.954 busy with 128-column tiles, ~0.91 with 80-column ones).
static double n_cost(long long n_ext, int nf) {
  const long long bn = gemm_bn(nf);
  return (double)((n_ext + bn - 1) / bn * bn) * (1.0 + 1.2 / nf);
}

int choose_nf(long long n_ext) {
  int best = kMaxNF;
  double best_cost = -1.0;
  for (int nf = kMaxNF; nf >= kMinNF; --nf) {
    const double cost = n_cost(n_ext, nf);
    if (best_cost < 0 || cost < best_cost) { best_cost = cost; best = nf; }
  }
  return best;
}

int split_n(int n_ext, NSegment seg[2], int granularity) {
  const int gr = granularity >= 16 ? 2 : 1;              // fragments per group
  const int gmax = kMaxNF / gr, gmin = (kMinNF + gr - 1) / gr;
  const int g = (n_ext + 8 * gr - 1) / (8 * gr);         // groups to cover
  if (g <= gmax) {
    seg[0] = {0, 1, gr * (g < gmin ? gmin : g)};
    return 1;
  }
  const int k = (g + gmax - 1) / gmax;                   // fewest tiles
  const int lo = g / k, nhi = g % k;                     // nhi tiles of lo+1 groups, the rest lo  (lo >= gmin)
  if (nhi == 0) {
    seg[0] = {0, k, gr * lo};
    return 1;
  }
  seg[0] = {0, nhi, gr * (lo + 1)};
  seg[1] = {nhi * gemm_bn(gr * (lo + 1)), k - nhi, gr * lo};
  return 2;
}

void choose_m_tile(int m1_ext, int m2_ext, int* tp, int* tq_log2) {
  long long best_cost = -1;
  for (int lg = 7; lg >= 3; --lg) {   // tq = 128 ... 8 (a TMA sub-box of tq rows must span whole 1 KiB swizzle atoms)
    const int tq = 1 << lg, tpp = kBM / tq;
    const long long cost = (long long)round_up_i(m1_ext, tpp) * round_up_i(m2_ext, tq);
    if (best_cost < 0 || cost < best_cost) { best_cost = cost; *tp = tpp; *tq_log2 = lg; }
  }
}

int split_m(int m1_ext, int m2_ext, MSegment seg[2]) {
  long long best = -1;
  int nbest = 0;
  for (int lg = 7; lg >= 3; --lg) {
    const int tq = 1 << lg, tp = kBM / tq;
    const int main_tiles = m1_ext / tp, r = m1_ext - main_tiles * tp;
    long long cost = (long long)main_tiles * tp * round_up_i(m2_ext, tq);
    MSegment cand[2];
    int n = 0;
    if (main_tiles > 0) cand[n++] = {0, main_tiles, tp, lg};
    if (r > 0) {
      int stp = 0, slg = 0;
      choose_m_tile(r, m2_ext, &stp, &slg);
      cost += (long long)round_up_i(r, stp) * round_up_i(m2_ext, 1 << slg);
      cand[n++] = {main_tiles * tp, ceil_div(r, stp), stp, slg};
    }
    if (best < 0 || cost < best) {
      best = cost;
      nbest = n;
      for (int k = 0; k < n; ++k) seg[k] = cand[k];
    }
  }
  return nbest;
}

template <int NF, bool kStaged, bool kTail>
static int launch_nf(const CUtensorMap& tmA, const CUtensorMap& tmAT, const CUtensorMap& tmB,
                     const GemmParams& prm, int grid, cudaStream_t stream) {
  // the > 48 KiB dynamic shared memory opt-in is a per-device function attribute
  static bool attr_set[64] = {};
  int dev = 0;
  BQC_CUDA_OK(cudaGetDevice(&dev));
  if (dev < 0 || dev >= 64 || !attr_set[dev]) {
    BQC_CUDA_OK(cudaFuncSetAttribute(gemm_nt_kernel<NF, kStaged, kTail>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                     gemm_smem_bytes(NF, kStaged)));
    if (dev >= 0 && dev < 64) attr_set[dev] = true;
  }
  gemm_nt_kernel<NF, kStaged, kTail><<<grid, kGemmThreads, gemm_smem_bytes(NF, kStaged), stream>>>(tmA, tmAT, tmB, prm);
  count_launch();
  BQC_CUDA_OK(cudaGetLastError());
  return BQC_OK;
}

int launch_gemm_nt(int nf, const CUtensorMap& tmA, const CUtensorMap& tmAT, const CUtensorMap& tmB,
                   const GemmParams& prm, cudaStream_t stream) {
  const long long total = (long long)prm.ntasks * prm.tiles_m1 * prm.tiles_m2 * prm.tiles_n;
  if (total <= 0) return BQC_OK;
  if (total >= (1LL << 31)) {
    set_error(BQC_ERR_INVALID_SIZE, "launch_gemm_nt: %lld tiles in one launch (limit 2^31)", total);
    return BQC_ERR_INVALID_SIZE;
  }
  const int sms = device_sm_count();
  if (sms <= 0) {
    set_error(BQC_ERR_CUDA, "no CUDA device");
    return BQC_ERR_CUDA;
  }
  const int grid = (int)(total < sms ? total : sms);
  // blocked (F-layout) output goes through the shared-memory staging tile and bulk stores; it needs whole
  // 8-row groups of one m1 per fragment row block, i.e. tq >= 8 (always true: choose_m_tile / split_m)
  const bool staged = prm.out_mode == 1;
  if (staged && prm.tq_log2 < 3) {
    set_error(BQC_ERR_INVALID_OPTION, "launch_gemm_nt: blocked output needs tq >= 8");
    return BQC_ERR_INVALID_OPTION;
  }
  // The K-tail instantiation halves the last stage of every term when it holds <= 8 valid columns; its peeled
  // stage loop runs the full stages as fast as the plain one (measured), so it is used whenever it applies.
  const bool ktail = prm.ktail8 != 0;
  switch (nf) {
#define BQC_NF_CASE(n)                                                                            \
  case n:                                                                                         \
    if (ktail)                                                                                    \
      return staged ? launch_nf<n, true, true>(tmA, tmAT, tmB, prm, grid, stream)                 \
                    : launch_nf<n, false, true>(tmA, tmAT, tmB, prm, grid, stream);               \
    return staged ? launch_nf<n, true, false>(tmA, tmAT, tmB, prm, grid, stream)                  \
                  : launch_nf<n, false, false>(tmA, tmAT, tmB, prm, grid, stream)
    BQC_NF_CASE(4); BQC_NF_CASE(5); BQC_NF_CASE(6); BQC_NF_CASE(7); BQC_NF_CASE(8); BQC_NF_CASE(9);
    BQC_NF_CASE(10); BQC_NF_CASE(11); BQC_NF_CASE(12); BQC_NF_CASE(13); BQC_NF_CASE(14); BQC_NF_CASE(15);
    BQC_NF_CASE(16);
#undef BQC_NF_CASE
  }
  set_error(BQC_ERR_INVALID_OPTION, "launch_gemm_nt: unsupported nf %d", nf);
  return BQC_ERR_INVALID_OPTION;
}

}  // namespace bqc
