// mp2.cu — closed-shell DF-MP2 energy (§2.3 Eq. (1)).
//
//   J_ij[a,b] = (ia|jb) = sum_Q B_ov[Q,i,a] B_ov[Q,j,b]
//   e_ij      = sum_ab J_ij[a,b] (2 J_ij[a,b] - J_ij[b,a]) / (eps_i + eps_j - eps_a - eps_b)
//   E_MP2     = sum_{i<=j} (2 - d_ij) e_ij
//
// One block of occupied rows [i0, i1) at a time: the (ov|ov) block
//     Jblk[(i - i0) v + a][(j - i0) v + b],   i0 <= i < i1,  i0 <= j < o
// is one "NT" product of the K-major copy Bt_ov[(i,a)][Q] with itself, run on the library's TMA + DMMA
// tile-GEMM engine (gemm_nt.cuh); the whole (ov|ov) tensor (11.6 GB at config 5) is never stored.
// mp2_pair_kernel then reads every element of the pairs i <= j exactly once — a CTA owns a pair of
// mirror-image 32 x 32 tiles (A,B), (B,A) of one J_ij, so J[a,b] and J[b,a] meet in shared memory — with the
// denominator computed in registers (no D tensor).  Fixed-order reductions throughout.
#include <limits.h>
#include <math.h>
#include <string.h>

#include <algorithm>
#include <vector>

#include "gemm_nt.cuh"
#include "kernels.cuh"

namespace bqc {

namespace {

constexpr int kMT = 32;            // tile edge of the pair-energy kernel
constexpr int kMThreads = 256;     // 32 x 8 threads, 4 tile rows each

static thread_local double g_mp2_profile[6] = {0, 0, 0, 0, 0, 0};

struct Mp2Args {
  const double* J;          // block buffer, row pitch ld
  const double* eps_occ;
  const double* eps_vir;
  const int* tiles;         // [ntp] packed A | B << 16, A <= B
  double* partial;          // [rows_blk * ncol_occ][ntp]
  long long ld;
  int i0, ni, o, v, ntp;
};

// Pair slot p of a block of ni rows x nj columns counts the pairs il <= jl row by row: row il holds nj - il of
// them.  Returns il and jl (ni is at most a few dozen: a short loop).
__device__ __forceinline__ void pair_of_slot(int p, int nj, int* il, int* jl) {
  int r = 0;
  while (p >= nj - r) { p -= nj - r; ++r; }
  *il = r;
  *jl = r + p;
}
static long long pair_slots(int ni, int nj) { return (long long)ni * nj - (long long)ni * (ni - 1) / 2; }

// grid: (pair slot il <= jl of the block, tile pair): only the pairs i <= j are launched
__global__ void __launch_bounds__(kMThreads) mp2_pair_kernel(const Mp2Args a) {
  __shared__ double t1[kMT][kMT + 1];   // J[a in A][b in B]
  __shared__ double t2[kMT][kMT + 1];   // J[a in B][b in A]
  __shared__ double red[kMThreads / 32];
  int il, jl;
  pair_of_slot(blockIdx.x, a.o - a.i0, &il, &jl);
  const int packed = a.tiles[blockIdx.y];
  const int A = packed & 0xffff, B = packed >> 16;
  const int v = a.v;
  const double* Jp = a.J + (long long)il * v * a.ld + (long long)jl * v;
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
  const bool diag = (A == B);
#pragma unroll
  for (int r = 0; r < kMT; r += 8) {
    const int ra = A * kMT + r + ty, cb = B * kMT + tx;
    t1[r + ty][tx] = (ra < v && cb < v) ? __ldg(Jp + (long long)ra * a.ld + cb) : 0.0;
    if (!diag) {
      const int rb = B * kMT + r + ty, ca = A * kMT + tx;
      t2[r + ty][tx] = (rb < v && ca < v) ? __ldg(Jp + (long long)rb * a.ld + ca) : 0.0;
    }
  }
  __syncthreads();
  const double eij = a.eps_occ[a.i0 + il] + a.eps_occ[a.i0 + jl];
  const int gb = B * kMT + tx;
  const double eb = gb < v ? __ldg(a.eps_vir + gb) : 0.0;
  double acc = 0.0;
#pragma unroll
  for (int r = 0; r < kMT; r += 8) {
    const int la = r + ty, ga = A * kMT + la;
    if (ga < v && gb < v) {
      const double d = eij - __ldg(a.eps_vir + ga) - eb;      // D_ij^ab = D_ij^ba
      const double x = t1[la][tx];                            // J[a,b]
      const double y = diag ? t1[tx][la] : t2[tx][la];        // J[b,a]
      // off-diagonal tile pair: the (a,b) and (b,a) terms of Eq. (1) together; diagonal tile: the (a,b) term
      const double num = diag ? x * (2.0 * x - y) : 2.0 * (x * x + y * y - x * y);
      acc += num / d;
    }
  }
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, off);
  if (tx == 0) red[ty] = acc;
  __syncthreads();
  if (threadIdx.x == 0) {
    double s = 0.0;
#pragma unroll
    for (int w = 0; w < kMThreads / 32; ++w) s += red[w];
    a.partial[(size_t)blockIdx.x * a.ntp + blockIdx.y] = s;
  }
}

// one CTA per pair slot of the block: e_ij = sum_tilepairs partial (fixed tree); writes the pair matrix (both
// triangles, unweighted) and the weighted entry (2 - d_ij) e_ij of the final-sum array
__global__ void mp2_reduce_pairs_kernel(const double* __restrict__ partial, int ntp, int i0, int o,
                                        double* __restrict__ e_pair, double* __restrict__ e_w) {
  __shared__ double red[128];
  int il, jl;
  pair_of_slot(blockIdx.x, o - i0, &il, &jl);
  const double* p = partial + (size_t)blockIdx.x * ntp;
  double s = 0.0;
  for (int n = threadIdx.x; n < ntp; n += 128) s += p[n];
  red[threadIdx.x] = s;
  __syncthreads();
  for (int off = 64; off > 0; off >>= 1) {
    if (threadIdx.x < off) red[threadIdx.x] += red[threadIdx.x + off];
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    const int i = i0 + il, j = i0 + jl;
    e_pair[(size_t)i * o + j] = red[0];
    e_pair[(size_t)j * o + i] = red[0];
    e_w[(size_t)i * o + j] = (i == j ? 1.0 : 2.0) * red[0];
  }
}

int auto_block(int o, int v) {
  const double per_i = (double)v * o * v * 8.0;
  int bi = (int)floor(2.0 * 1073741824.0 / per_i);
  return std::max(1, std::min(bi, o));
}

int resolve_block(int o, int v, const bqc_mp2_opts* opts, int* bi) {
  const int b = opts ? opts->occ_block : 0;
  if (b < 0) {
    set_error(BQC_ERR_INVALID_OPTION, "mp2 occ_block %d < 0", b);
    return BQC_ERR_INVALID_OPTION;
  }
  *bi = b > 0 ? std::min(b, o) : auto_block(o, v);
  return BQC_OK;
}

struct Mp2Layout {
  size_t off_bt = 0, off_jblk = 0, off_partial = 0, off_epair = 0, off_ew = 0, off_esum = 0, off_tiles = 0,
         off_task = 0, total = 0;
};

Mp2Layout mp2_layout(int o, int v, int Xp, int Bi, int ntp) {
  Mp2Layout L;
  size_t off = 0;
  auto take = [&](size_t bytes) { size_t r = off; off = round_up(off + (bytes ? bytes : 8), 1024); return r; };
  L.off_bt = take((size_t)o * v * Xp * 8);                    // Bt_ov
  L.off_jblk = take((size_t)Bi * v * ((size_t)o * v) * 8);    // (ov|ov) block
  L.off_partial = take((size_t)Bi * o * ntp * 8);
  L.off_epair = take((size_t)o * o * 8);
  L.off_ew = take((size_t)o * o * 8);
  L.off_esum = take(64);
  L.off_tiles = take((size_t)ntp * 4);
  L.off_task = take(sizeof(GemmTask));
  L.total = off;
  return L;
}

struct Scratch {
  std::vector<void*> ptrs;
  std::vector<cudaEvent_t> evs;
  ~Scratch() {
    for (void* p : ptrs) cudaFree(p);
    for (cudaEvent_t e : evs) cudaEventDestroy(e);
  }
  int alloc(void** p, size_t bytes, const char* what) {
    cudaError_t e = cudaMalloc(p, bytes ? bytes : 8);
    if (e != cudaSuccess) {
      cudaGetLastError();
      set_error(BQC_ERR_WORKSPACE, "cudaMalloc of %zu bytes (%s) failed: %s", bytes, what, cudaGetErrorString(e));
      return BQC_ERR_WORKSPACE;
    }
    ptrs.push_back(*p);
    return BQC_OK;
  }
  int mark(cudaStream_t s) {
    cudaEvent_t e;
    BQC_CUDA_OK(cudaEventCreate(&e));
    evs.push_back(e);
    BQC_CUDA_OK(cudaEventRecord(e, s));
    return BQC_OK;
  }
};

}  // namespace

static int mp2_impl(int o, int v, int X, const double* eps_occ, const double* eps_vir, const double* B_ov,
                    const bqc_mp2_opts* opts, double* e_total_host, double* e_pair_dev, cudaStream_t s) {
  clear_error();
  if (!e_total_host) {
    set_error(BQC_ERR_NULL_POINTER, "e_total_host is NULL");
    return BQC_ERR_NULL_POINTER;
  }
  BQC_TRY(check_sizes(o, v, X));
  BQC_TRY(check_device());
  BQC_TRY(check_device_ptr(eps_occ, "eps_occ"));
  BQC_TRY(check_device_ptr(eps_vir, "eps_vir"));
  BQC_TRY(check_device_ptr(B_ov, "B_ov"));
  if (e_pair_dev) BQC_TRY(check_device_ptr(e_pair_dev, "e_pair_dev"));
  int Bi = 0;
  BQC_TRY(resolve_block(o, v, opts, &Bi));
  const int sc = (opts && opts->shard_count > 0) ? opts->shard_count : 1;
  const int sr = opts ? opts->shard_rank : 0;
  if (sr < 0 || sr >= sc) {
    set_error(BQC_ERR_INVALID_OPTION, "shard_rank %d outside [0,%d)", sr, sc);
    return BQC_ERR_INVALID_OPTION;
  }
  const bool prof = opts && (opts->flags & BQC_T_FLAG_PROFILE);
  {
    std::vector<double> eo(o), ev(v);
    BQC_CUDA_OK(cudaMemcpyAsync(eo.data(), eps_occ, (size_t)o * 8, cudaMemcpyDeviceToHost, s));
    BQC_CUDA_OK(cudaMemcpyAsync(ev.data(), eps_vir, (size_t)v * 8, cudaMemcpyDeviceToHost, s));
    BQC_CUDA_OK(cudaStreamSynchronize(s));
    const double emax = *std::max_element(eo.begin(), eo.end());
    const double vmin = *std::min_element(ev.begin(), ev.end());
    if (!(2.0 * emax - 2.0 * vmin < 0.0)) {
      set_error(BQC_ERR_DENOMINATOR, "2*max(eps_occ)=%g - 2*min(eps_vir)=%g >= 0: denominators may vanish",
                2.0 * emax, 2.0 * vmin);
      return BQC_ERR_DENOMINATOR;
    }
  }

  const int Xp = round_up_i(X, 16);
  const int nt = ceil_div(v, kMT), ntp = nt * (nt + 1) / 2;
  Scratch sc_mem;
  // one workspace block: the caller's (opts->workspace) or one cudaMalloc freed before return
  const Mp2Layout L = mp2_layout(o, v, Xp, Bi, ntp);
  uint8_t* ws = nullptr;
  if (opts && opts->workspace) {
    if (opts->workspace_bytes < L.total || (reinterpret_cast<uintptr_t>(opts->workspace) & 255)) {
      set_error(BQC_ERR_WORKSPACE, "mp2 workspace of %zu bytes (need %zu, 256-byte aligned)", opts->workspace_bytes,
                L.total);
      return BQC_ERR_WORKSPACE;
    }
    BQC_TRY(check_device_ptr(opts->workspace, "opts->workspace"));
    ws = static_cast<uint8_t*>(opts->workspace);
  } else {
    BQC_TRY(sc_mem.alloc((void**)&ws, L.total, "mp2 workspace"));
  }
  double* bt = reinterpret_cast<double*>(ws + L.off_bt);
  double* jblk = reinterpret_cast<double*>(ws + L.off_jblk);
  double* partial = reinterpret_cast<double*>(ws + L.off_partial);
  double* e_pair = reinterpret_cast<double*>(ws + L.off_epair);
  double* e_w = reinterpret_cast<double*>(ws + L.off_ew);
  double* e_sum = reinterpret_cast<double*>(ws + L.off_esum);
  int* tiles = reinterpret_cast<int*>(ws + L.off_tiles);
  GemmTask* task_dev = reinterpret_cast<GemmTask*>(ws + L.off_task);

  int nlaunch = 0;
  if (prof) BQC_TRY(sc_mem.mark(s));   // evs[0]: begin
  {
    std::vector<int> tl;
    for (int A = 0; A < nt; ++A)
      for (int B = A; B < nt; ++B) tl.push_back(A | (B << 16));
    BQC_CUDA_OK(cudaMemcpyAsync(tiles, tl.data(), tl.size() * 4, cudaMemcpyHostToDevice, s));
    GemmTask task;
    memset(&task, 0, sizeof(task));
    task.nterms = 1;
    BQC_CUDA_OK(cudaMemcpyAsync(task_dev, &task, sizeof(task), cudaMemcpyHostToDevice, s));
    BQC_CUDA_OK(cudaStreamSynchronize(s));   // host vectors go out of scope
  }
  BQC_CUDA_OK(cudaMemsetAsync(e_pair, 0, (size_t)o * o * 8, s));
  BQC_CUDA_OK(cudaMemsetAsync(e_w, 0, (size_t)o * o * 8, s));
  BQC_TRY(launch_transpose_pad(B_ov, (long long)o * v, 0, (long long)o * v, bt, X, Xp, 0, 0, s));   // Bt_ov[(i,a)][Q], zero-padded to Xp
  ++nlaunch;

  // The (ov|ov) sub-launches of a block alternate between the caller's stream and a helper stream: each is a
  // persistent one-CTA-per-SM kernel of ~12 waves of tiles, so in one stream the partly filled last wave of every
  // sub-launch (7 % of the time at config 5) would idle; on two streams the next sub-launch fills it.
  struct Helper {
    cudaStream_t s2 = nullptr;
    cudaEvent_t ready = nullptr, done = nullptr;
    ~Helper() {
      if (ready) cudaEventDestroy(ready);
      if (done) cudaEventDestroy(done);
      if (s2) cudaStreamDestroy(s2);
    }
  } hp;
  BQC_CUDA_OK(cudaStreamCreateWithFlags(&hp.s2, cudaStreamNonBlocking));
  BQC_CUDA_OK(cudaEventCreateWithFlags(&hp.ready, cudaEventDisableTiming));
  BQC_CUDA_OK(cudaEventCreateWithFlags(&hp.done, cudaEventDisableTiming));

  int ngemm = 0;
  const int nblk = ceil_div(o, Bi);
  for (int b = 0; b < nblk; ++b) {
    if (b % sc != sr) continue;
    const int i0 = b * Bi, i1 = std::min(o, i0 + Bi);
    const long long ld = (long long)(o - i0) * v;
    // The (ov|ov) rows of the block are formed `grows` occupied orbitals at a time, each sub-launch covering only
    // the columns j >= its first row: the pairs j < i that a rectangular block GEMM would also compute shrink
    // from ~15 % of the work (18-row blocks at config 5) to ~2 %.  grows keeps >= ~8 waves of tiles per launch.
    const int grows = std::max(2, std::min(Bi, (int)ceil(3.9e7 / ((double)o * v * v))));
    if (prof) BQC_TRY(sc_mem.mark(s));
    // the helper stream may write the block buffer once the previous block's pair kernel has read it
    BQC_CUDA_OK(cudaEventRecord(hp.ready, s));
    BQC_CUDA_OK(cudaStreamWaitEvent(hp.s2, hp.ready, 0));
    int sub = 0;
    for (int g0 = i0; g0 < i1; g0 += grows) {
      cudaStream_t sg = (sub++ & 1) ? hp.s2 : s;
      const int g1 = std::min(i1, g0 + grows);
      const int M = (g1 - g0) * v;
      const long long N = (long long)(o - g0) * v;
      const int nf = choose_nf(N);
      CUtensorMap tA, tB;
      const double* base = bt + (size_t)g0 * v * Xp;   // rows (g0, 0) onwards; 128-byte aligned (Xp % 16 == 0)
      const unsigned long long dA[4] = {(unsigned long long)Xp, (unsigned long long)M, 1, 1};
      const unsigned long long sA[4] = {8, (unsigned long long)Xp * 8, (unsigned long long)Xp * 8 * M,
                                        (unsigned long long)Xp * 8 * M};
      BQC_TRY(make_tensor_map_f64(&tA, base, dA, sA, 128, 1));
      const unsigned long long dB[4] = {(unsigned long long)Xp, (unsigned long long)N, 1, 1};
      const unsigned long long sB[4] = {8, (unsigned long long)Xp * 8, (unsigned long long)Xp * 8 * N,
                                        (unsigned long long)Xp * 8 * N};
      BQC_TRY(make_tensor_map_f64(&tB, base, dB, sB, gemm_bn(nf), 1));
      GemmParams prm;
      memset(&prm, 0, sizeof(prm));
      prm.ntasks = 1;
      prm.tp = 1; prm.tq_log2 = 7;
      prm.tiles_m1 = 1;
      prm.tiles_m2 = ceil_div(M, kBM);
      prm.tiles_n = (int)((N + gemm_bn(nf) - 1) / gemm_bn(nf));
      prm.m1_ext = 1; prm.m2_ext = M; prm.n_ext = (int)N;
      prm.kiters = Xp / kBK;
      prm.ktail8 = (X - (prm.kiters - 1) * kBK) <= 8;
      prm.out_mode = 0;
      prm.n2_ext = INT_MAX;
      prm.sM1 = 0; prm.sM2 = ld; prm.sN1 = 0; prm.sN2 = 1;
      prm.tasks = task_dev;
      // element (row (i - g0) v + a, column (j - g0) v + b) of this sub-launch -> Jblk[(i - i0) v + a][(j - i0) v + b]
      prm.C = jblk + (long long)(g0 - i0) * v * ld + (long long)(g0 - i0) * v;
      BQC_TRY(launch_gemm_nt(nf, tA, tA, tB, prm, sg));
      ++nlaunch;
    }
    BQC_CUDA_OK(cudaEventRecord(hp.done, hp.s2));
    BQC_CUDA_OK(cudaStreamWaitEvent(s, hp.done, 0));
    if (prof) BQC_TRY(sc_mem.mark(s));
    ++ngemm;

    Mp2Args a;
    a.J = jblk; a.eps_occ = eps_occ; a.eps_vir = eps_vir; a.tiles = tiles; a.partial = partial;
    a.ld = ld; a.i0 = i0; a.ni = i1 - i0; a.o = o; a.v = v; a.ntp = ntp;
    const int nslots = (int)pair_slots(i1 - i0, o - i0);
    mp2_pair_kernel<<<dim3(nslots, ntp), kMThreads, 0, s>>>(a);
    count_launch();
    BQC_CUDA_OK(cudaGetLastError());
    mp2_reduce_pairs_kernel<<<nslots, 128, 0, s>>>(partial, ntp, i0, o, e_pair, e_w);
    count_launch();
    BQC_CUDA_OK(cudaGetLastError());
    if (prof) BQC_TRY(sc_mem.mark(s));
    nlaunch += 2;
  }
  BQC_TRY(launch_final_sum(e_w, (long long)o * o, e_sum, s));
  ++nlaunch;
  if (prof) BQC_TRY(sc_mem.mark(s));   // end
  if (e_pair_dev) BQC_CUDA_OK(cudaMemcpyAsync(e_pair_dev, e_pair, (size_t)o * o * 8, cudaMemcpyDeviceToDevice, s));
  BQC_CUDA_OK(cudaMemcpyAsync(e_total_host, e_sum, 8, cudaMemcpyDeviceToHost, s));
  BQC_CUDA_OK(cudaStreamSynchronize(s));
  g_mp2_profile[5] = nlaunch;
  if (prof) {
    double gemm_ms = 0, en_ms = 0;
    float ms = 0.f;
    for (int n = 0; n < ngemm; ++n) {
      BQC_CUDA_OK(cudaEventElapsedTime(&ms, sc_mem.evs[1 + 3 * n], sc_mem.evs[2 + 3 * n]));
      gemm_ms += ms;
      BQC_CUDA_OK(cudaEventElapsedTime(&ms, sc_mem.evs[2 + 3 * n], sc_mem.evs[3 + 3 * n]));
      en_ms += ms;
    }
    BQC_CUDA_OK(cudaEventElapsedTime(&ms, sc_mem.evs.front(), sc_mem.evs.back()));
    g_mp2_profile[0] = gemm_ms; g_mp2_profile[1] = ngemm;
    g_mp2_profile[2] = en_ms;   g_mp2_profile[3] = 2.0 * ngemm;
    g_mp2_profile[4] = ms;
  }
  return BQC_OK;
}

}  // namespace bqc

using namespace bqc;

extern "C" {

double bqc_mp2_flops(int nocc, int nvir, int naux) {
  if (nocc <= 0 || nvir <= 0 || naux <= 0) return 0.0;
  return 0.5 * nocc * (nocc + 1.0) * 2.0 * (double)nvir * nvir * naux;
}

size_t bqc_mp2_workspace_bytes(int nocc, int nvir, int naux, const bqc_mp2_opts* opts) {
  clear_error();
  if (check_sizes(nocc, nvir, naux) != BQC_OK) return 0;
  int bi = 0;
  if (resolve_block(nocc, nvir, opts, &bi) != BQC_OK) return 0;
  const int nt = ceil_div(nvir, kMT);
  return mp2_layout(nocc, nvir, round_up_i(naux, 16), bi, nt * (nt + 1) / 2).total;
}

int bqc_mp2_plan_occ_block(int nocc, int nvir, int naux, const bqc_mp2_opts* opts) {
  clear_error();
  if (check_sizes(nocc, nvir, naux) != BQC_OK) return -1;
  int bi = 0;
  if (resolve_block(nocc, nvir, opts, &bi) != BQC_OK) return -1;
  return bi;
}

int bqc_mp2_last_profile(double* out, int n) {
  if (!out || n <= 0) return 0;
  const int m = n < 6 ? n : 6;
  for (int i = 0; i < m; ++i) out[i] = g_mp2_profile[i];
  return m;
}

int bqc_mp2_energy_ex(int nocc, int nvir, int naux, const double* eps_occ, const double* eps_vir,
                      const double* B_ov, const bqc_mp2_opts* opts, double* e_total_host, double* e_pair_dev,
                      void* stream) {
  return mp2_impl(nocc, nvir, naux, eps_occ, eps_vir, B_ov, opts, e_total_host, e_pair_dev,
                  static_cast<cudaStream_t>(stream));
}

double bqc_mp2_energy(int nocc, int nvir, int naux, const double* eps_occ, const double* eps_vir,
                      const double* B_ov, void* stream) {
  double e = 0.0;
  const int rc = bqc_mp2_energy_ex(nocc, nvir, naux, eps_occ, eps_vir, B_ov, nullptr, &e, nullptr, stream);
  return rc == BQC_OK ? e : nan("");
}

int bqc_mp2_energy_host(int nocc, int nvir, int naux, const double* eps_occ, const double* eps_vir,
                        const double* B_ov, const bqc_mp2_opts* opts, double* e_total_host, double* e_pair_host,
                        size_t* h2d_bytes, size_t* d2h_bytes, void* stream_v) {
  clear_error();
  cudaStream_t stream = static_cast<cudaStream_t>(stream_v);
  BQC_TRY(check_sizes(nocc, nvir, naux));
  const void* ptrs[3] = {eps_occ, eps_vir, B_ov};
  const char* names[3] = {"eps_occ", "eps_vir", "B_ov"};
  const size_t o = nocc, v = nvir, X = naux;
  const size_t elems[3] = {o, v, X * o * v};
  for (int n = 0; n < 3; ++n)
    if (!ptrs[n]) {
      set_error(BQC_ERR_NULL_POINTER, "%s is NULL", names[n]);
      return BQC_ERR_NULL_POINTER;
    }
  if (!e_total_host) {
    set_error(BQC_ERR_NULL_POINTER, "e_total_host is NULL");
    return BQC_ERR_NULL_POINTER;
  }
  size_t total = 0, offs[3];
  for (int n = 0; n < 3; ++n) { offs[n] = total; total += round_up(elems[n] * 8, 256); }
  const size_t off_pair = total;
  total += round_up(o * o * 8, 256);
  uint8_t* dev = nullptr;
  {
    cudaError_t e = cudaMalloc(&dev, total);
    if (e != cudaSuccess) {
      cudaGetLastError();
      set_error(BQC_ERR_WORKSPACE, "cudaMalloc of %zu input bytes failed: %s", total, cudaGetErrorString(e));
      return BQC_ERR_WORKSPACE;
    }
  }
  int rc = BQC_OK;
  size_t h2d = 0;
  for (int n = 0; n < 3 && rc == BQC_OK; ++n) {
    cudaError_t e = cudaMemcpyAsync(dev + offs[n], ptrs[n], elems[n] * 8, cudaMemcpyHostToDevice, stream);
    if (e != cudaSuccess) {
      set_error(BQC_ERR_CUDA, "H2D copy of %s failed: %s", names[n], cudaGetErrorString(e));
      rc = BQC_ERR_CUDA;
    }
    h2d += elems[n] * 8;
  }
  if (rc == BQC_OK) {
    auto D = [&](int n) { return reinterpret_cast<const double*>(dev + offs[n]); };
    rc = bqc_mp2_energy_ex(nocc, nvir, naux, D(0), D(1), D(2), opts, e_total_host,
                           e_pair_host ? reinterpret_cast<double*>(dev + off_pair) : nullptr, stream);
  }
  size_t d2h = 8;
  if (rc == BQC_OK && e_pair_host) {
    cudaError_t e = cudaMemcpyAsync(e_pair_host, dev + off_pair, o * o * 8, cudaMemcpyDeviceToHost, stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(stream);
    if (e != cudaSuccess) {
      set_error(BQC_ERR_CUDA, "D2H copy of e_pair failed: %s", cudaGetErrorString(e));
      rc = BQC_ERR_CUDA;
    }
    d2h += o * o * 8;
  }
  cudaFree(dev);
  if (h2d_bytes) *h2d_bytes = h2d;
  if (d2h_bytes) *d2h_bytes = d2h;
  return rc;
}

}  // extern "C"
