// t_energy.cu — planner, triplet-block scheduler and C ABI of libbqc_t.so.
//
// How W is built:
//   augmented slab   I~_x[p,q,kappa] : kappa <  v      -> (x p|q d)                 (DF slab former, a1)
//                                      kappa = v + l   -> -t2[x,l,p,q]              (hole columns)
//   augmented pair   B~_zy[r,kappa]  : kappa <  v      -> t2[z,y,r,d]
//                                      kappa = v + l   -> (z r|y l)                 (DF slab former, a1)
//   F(x,y,z)[p,q,r] = sum_kappa I~_x[p,q,kappa] B~_zy[r,kappa] + sum_kappa I~_y[q,p,kappa] B~_zx[r,kappa]
//   W_ijk[a,b,c]    = F(i,j,k)[a,b,c] + F(i,k,j)[a,c,b] + F(j,k,i)[b,c,a]          (= PAPER.md Eq. (2), G1/G5)
// i.e. the six particle and six hole contractions of Eq. (2) become six K = v+o tile-GEMM terms.
#include <limits.h>
#include <math.h>
#include <stdarg.h>
#include <string.h>

#include <algorithm>
#include <vector>

#include "gemm_nt.cuh"
#include "kernels.cuh"

namespace bqc {

// ------------------------------------------------------------------ error state
static thread_local int g_err = BQC_OK;
static thread_local char g_detail[512] = "";

void set_error(int code, const char* fmt, ...) {
  g_err = code;
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_detail, sizeof(g_detail), fmt, ap);
  va_end(ap);
}
void clear_error() {
  g_err = BQC_OK;
  g_detail[0] = 0;
}

static thread_local double g_profile[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};
static thread_local long long g_launches = 0;
void count_launch(int n) { g_launches += n; }

namespace {

// ------------------------------------------------------------------ plan
struct Plan {
  int o = 0, v = 0, X = 0;
  std::vector<int> act;        // active occupied orbitals (sorted); triplets are drawn from these
  int na = 0;                  // act.size()
  int Xp = 0, Kp = 0;          // aux / (v+o) extents padded to multiples of 16
  int nbv = 0;                 // 8-blocks per virtual dimension
  size_t fsz = 0;              // doubles per blocked F array
  size_t slab_elems = 0;       // v*v*Kp
  int Bo = 0, nblk = 0, nsets = 0, nslots = 0;
  int nbatch = 0;              // triplets per W-builder launch
  int norbits = 0;
  int use_t1 = 1;
  int profile = 0;
  int shard_rank = 0, shard_count = 1;
  int shard_blocks = 0;        // BQC_T_FLAG_SHARD_BLOCKS
  // workspace offsets (bytes)
  size_t off_btvv = 0, off_btov = 0, off_btoo = 0, off_btil = 0, off_J = 0, off_slabs = 0, off_F = 0,
         off_partial = 0, off_etrip = 0, off_esum = 0, off_act = 0, off_orbits = 0, off_tasks = 0,
         off_trips = 0, total = 0;
  size_t max_tasks = 0, max_trips = 0;
};

size_t num_triplets(int o) { return (size_t)o * (o + 1) * (o + 2) / 6; }

size_t triplet_index(int o, int i, int j, int k) {
  // lexicographic rank of (i,j,k), i<=j<=k<o
  auto below = [&](int m) { return (size_t)m * (m + 1) * (m + 2) / 6; };   // #triplets over m orbitals
  // triplets whose first index < i: all triplets over o minus those over (o - i) shifted
  size_t r = below(o) - below(o - i);
  // first index == i, second index in [i, j): for second index s the third runs over (o - s) values
  const size_t n1 = (size_t)(o - i), n2 = (size_t)(o - j);
  r += n1 * (n1 + 1) / 2 - n2 * (n2 + 1) / 2;
  r += (size_t)(k - j);
  return r;
}

int resolve_window(int o, const bqc_t_opts* opts, int* lo, int* hi) {
  *lo = 0;
  *hi = o;
  if (opts && !(opts->occ_lo == 0 && opts->occ_hi == 0)) {
    *lo = opts->occ_lo;
    *hi = opts->occ_hi;
  }
  if (*lo < 0 || *hi > o || *lo >= *hi) {
    set_error(BQC_ERR_INVALID_OPTION, "occupied window [%d,%d) invalid for nocc=%d", *lo, *hi, o);
    return BQC_ERR_INVALID_OPTION;
  }
  return BQC_OK;
}

int auto_occ_block(int na, int v, int Kp) {
  // 4*Bo augmented slabs resident; keep them under ~24 GiB
  const double slab_bytes = (double)v * v * Kp * 8.0;
  int bo = (int)floor(24.0 * 1073741824.0 / (4.0 * slab_bytes));
  bo = std::max(1, std::min(bo, na));
  const int nblk = ceil_div(na, bo);
  return ceil_div(na, nblk);   // balanced blocks
}

// Non-diagonal triplets pi <= pj <= pk of block triple (I, J, K) over na orbitals in blocks of bo.
long long block_triple_work(int na, int bo, int I, int J, int K) {
  auto b0 = [&](int b) { return b * bo; };
  auto b1 = [&](int b) { return std::min(na, (b + 1) * bo); };
  long long n = 0;
  for (int pi = b0(I); pi < b1(I); ++pi)
    for (int pj = std::max(pi, b0(J)); pj < b1(J); ++pj) {
      const int k0 = std::max(pj, b0(K));
      n += std::max(0, b1(K) - k0);
      if (pi == pj && pj >= k0 && pj < b1(K)) --n;   // i = j = k contributes exactly 0 and is skipped
    }
  return n;
}

// BQC_T_FLAG_SHARD_BLOCKS: owner of every block triple I <= J <= K (numbered in loop order).  Largest block
// triples first, each to the least-loaded rank so far (ties: lower rank) — a deterministic function of
// (na, bo, shard_count), so every rank and the host helpers (bqc_t_flops, bqc_t_triplet_owner_ex) agree.
std::vector<int> deal_block_triples(int na, int bo, int shard_count, std::vector<long long>* load_out = nullptr) {
  const int nblk = ceil_div(na, bo);
  struct BT { long long work; int id; };
  std::vector<BT> bt;
  int id = 0;
  for (int I = 0; I < nblk; ++I)
    for (int J = I; J < nblk; ++J)
      for (int K = J; K < nblk; ++K) bt.push_back({block_triple_work(na, bo, I, J, K), id++});
  std::vector<int> owner(bt.size(), 0);
  std::vector<long long> load(shard_count, 0);
  std::stable_sort(bt.begin(), bt.end(), [](const BT& a, const BT& b) { return a.work > b.work; });
  for (const BT& t : bt) {
    int best = 0;
    for (int r = 1; r < shard_count; ++r)
      if (load[r] < load[best]) best = r;
    owner[t.id] = best;
    load[best] += t.work;
  }
  if (load_out) *load_out = load;
  return owner;
}

// Block size for a block-triple-sharded run: the largest Bo <= the memory-derived one whose deal is within
// 3 % of even (the slabs of a block are re-formed by every rank that owns one of its triples, so larger is
// cheaper); the best one found if none is.
int balanced_occ_block(int na, int bo_max, int shard_count) {
  int best_bo = bo_max;
  double best = -1.0;
  for (int bo = bo_max; bo >= 1; --bo) {
    if (bo < bo_max && ceil_div(na, bo) == ceil_div(na, bo + 1)) continue;   // same block count: skip
    std::vector<long long> load;
    deal_block_triples(na, bo, shard_count, &load);
    long long mx = 0, sum = 0;
    for (long long l : load) { mx = std::max(mx, l); sum += l; }
    if (sum == 0) return bo_max;
    const double imb = (double)mx * shard_count / (double)sum;
    if (best < 0 || imb < best - 1e-12) { best = imb; best_bo = bo; }
    if (imb <= 1.03) break;
    if (ceil_div(na, bo) > 64) break;   // enough block triples (> 45 000): stop searching
  }
  return best_bo;
}

int make_plan(Plan& P, int o, int v, int X, const std::vector<int>& act, const bqc_t_opts* opts) {
  P.o = o; P.v = v; P.X = X;
  P.act = act;
  P.na = (int)act.size();
  P.Xp = round_up_i(X, 16);
  P.Kp = round_up_i(v + o, 16);
  P.nbv = ceil_div(v, kVB);
  P.fsz = (size_t)P.nbv * P.nbv * P.nbv * (kVB * kVB * kVB);
  P.slab_elems = (size_t)v * v * P.Kp;
  P.norbits = (int)((long long)P.nbv * (P.nbv + 1) * (P.nbv + 2) / 6);
  P.use_t1 = !(opts && (opts->flags & BQC_T_FLAG_NO_T1));
  P.profile = (opts && (opts->flags & BQC_T_FLAG_PROFILE)) ? 1 : 0;
  P.shard_count = (opts && opts->shard_count > 0) ? opts->shard_count : 1;
  P.shard_rank = opts ? opts->shard_rank : 0;
  P.shard_blocks = (opts && (opts->flags & BQC_T_FLAG_SHARD_BLOCKS)) ? 1 : 0;
  if (P.shard_rank < 0 || P.shard_rank >= P.shard_count) {
    set_error(BQC_ERR_INVALID_OPTION, "shard_rank %d outside [0,%d)", P.shard_rank, P.shard_count);
    return BQC_ERR_INVALID_OPTION;
  }
  int bo = opts ? opts->occ_block : 0;
  if (bo < 0) {
    set_error(BQC_ERR_INVALID_OPTION, "occ_block %d < 0", bo);
    return BQC_ERR_INVALID_OPTION;
  }
  P.Bo = bo > 0 ? std::min(bo, P.na) : auto_occ_block(P.na, v, P.Kp);
  if (bo == 0 && P.shard_blocks && P.shard_count > 1) P.Bo = balanced_occ_block(P.na, P.Bo, P.shard_count);
  P.nblk = ceil_div(P.na, P.Bo);
  P.nsets = P.nblk == 1 ? 1 : 4;
  P.nslots = P.nsets * P.Bo;
  int nbatch = opts ? opts->max_batch : 0;
  if (nbatch < 0) {
    set_error(BQC_ERR_INVALID_OPTION, "max_batch %d < 0", nbatch);
    return BQC_ERR_INVALID_OPTION;
  }
  if (nbatch == 0) {
    const double per = 3.0 * (double)P.fsz * 8.0;
    nbatch = (int)floor(6.0 * 1073741824.0 / per);
  }
  P.nbatch = std::max(1, std::min(nbatch, 1024));

  // upper bounds for the schedule arrays: every active triplet once, + DF tasks
  size_t ntrip_act = (size_t)P.na * (P.na + 1) * (P.na + 2) / 6;
  P.max_trips = ntrip_act + 8;
  P.max_tasks = 3 * ntrip_act + 64 + (size_t)P.na * P.na * 2 + 4 * (size_t)P.na;

  size_t off = 0;
  auto take = [&](size_t bytes) { size_t r = off; off = round_up(off + bytes, 1024); return r; };
  P.off_btvv = take((size_t)v * v * P.Xp * 8);
  P.off_btov = take((size_t)o * v * P.Xp * 8);
  P.off_btoo = take((size_t)o * o * P.Xp * 8);
  P.off_btil = take((size_t)P.na * P.na * v * P.Kp * 8);
  P.off_J = take((size_t)P.na * P.na * v * v * 8);
  P.off_slabs = take((size_t)P.nslots * P.slab_elems * 8);
  P.off_F = take((size_t)P.nbatch * 3 * P.fsz * 8);
  P.off_partial = take((size_t)P.nbatch * P.norbits * 8);
  P.off_etrip = take(num_triplets(o) * 8);
  P.off_esum = take(64);
  P.off_act = take((size_t)P.na * 4);
  P.off_orbits = take((size_t)P.norbits * 4);
  P.off_tasks = take(P.max_tasks * sizeof(GemmTask));
  P.off_trips = take(P.max_trips * sizeof(TripletRec));
  P.total = off;
  return BQC_OK;
}

}  // namespace

// ------------------------------------------------------------------ argument checks (shared with mp2.cu)
int check_sizes(int o, int v, int X) {
  if (o <= 0 || v <= 0 || X <= 0) {
    set_error(BQC_ERR_INVALID_SIZE, "nocc=%d nvir=%d naux=%d must all be > 0", o, v, X);
    return BQC_ERR_INVALID_SIZE;
  }
  if (v > 1023 * kVB || o > 4096) {
    set_error(BQC_ERR_INVALID_SIZE, "nocc=%d nvir=%d exceed the supported range", o, v);
    return BQC_ERR_INVALID_SIZE;
  }
  return BQC_OK;
}

int check_device_ptr(const void* p, const char* name) {
  if (!p) {
    set_error(BQC_ERR_NULL_POINTER, "%s is NULL", name);
    return BQC_ERR_NULL_POINTER;
  }
  if (reinterpret_cast<uintptr_t>(p) & 7) {
    set_error(BQC_ERR_MISALIGNED, "%s is not 8-byte aligned", name);
    return BQC_ERR_MISALIGNED;
  }
  cudaPointerAttributes attr;
  cudaError_t e = cudaPointerGetAttributes(&attr, p);
  if (e != cudaSuccess) {
    cudaGetLastError();
    set_error(BQC_ERR_NOT_DEVICE_PTR, "%s: cudaPointerGetAttributes failed: %s", name, cudaGetErrorString(e));
    return BQC_ERR_NOT_DEVICE_PTR;
  }
  if (attr.type != cudaMemoryTypeDevice && attr.type != cudaMemoryTypeManaged) {
    set_error(BQC_ERR_NOT_DEVICE_PTR, "%s is not device memory", name);
    return BQC_ERR_NOT_DEVICE_PTR;
  }
  return BQC_OK;
}

int check_device() {
  int dev = 0;
  BQC_CUDA_OK(cudaGetDevice(&dev));
  int major = 0;
  BQC_CUDA_OK(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
  if (major != 10) {
    set_error(BQC_ERR_DEVICE, "device compute capability %d.x is not sm_100 (B200)", major);
    return BQC_ERR_DEVICE;
  }
  return BQC_OK;
}

namespace {

struct Inputs {
  const double *eps_occ, *eps_vir, *t1, *t2, *B_oo, *B_ov, *B_vv;
  const double* f_ov = nullptr;   // optional occupied-virtual Fock block (bqc_t_opts.f_ov)
};

// ------------------------------------------------------------------ run context
struct Ctx {
  Plan P;
  Inputs in;
  uint8_t* ws = nullptr;
  bool own_ws = false;
  cudaStream_t s_main = nullptr, s_form = nullptr;
  cudaEvent_t ev_formed[4] = {}, ev_free[4] = {}, ev_fork = nullptr, ev_join = nullptr;
  bool ev_free_valid[4] = {};
  int set_block[4] = {-1, -1, -1, -1};
  // F-GEMM configuration
  MSegment f_mseg[2];                // row segments of the F GEMM (split_m): main tiles + remainder strip
  int f_nmseg = 0;
  NSegment f_seg[2];                 // column segments of the F GEMM (split_n): exact cover of v up to 16
  int f_nseg = 0;
  CUtensorMap tm_slab[2], tm_slabT[2], tm_btil[2];
  // host schedule
  std::vector<GemmTask> tasks;
  std::vector<TripletRec> trips;
  // BQC_T_FLAG_PROFILE: timing events, [3n] before W builder, [3n+1] after it, [3n+2] after the energy kernels
  std::vector<cudaEvent_t> prof_main;
  std::vector<cudaEvent_t> prof_form;   // [2n], [2n+1] around each slab-block formation
  cudaEvent_t prof_begin = nullptr, prof_prepared = nullptr, prof_end = nullptr;
  int prof_mark(std::vector<cudaEvent_t>& v, cudaStream_t s) {
    cudaEvent_t e;
    BQC_CUDA_OK(cudaEventCreate(&e));
    v.push_back(e);
    BQC_CUDA_OK(cudaEventRecord(e, s));
    return BQC_OK;
  }

  double* d(size_t off) const { return reinterpret_cast<double*>(ws + off); }
  double* btvv() const { return d(P.off_btvv); }
  double* btov() const { return d(P.off_btov); }
  double* btoo() const { return d(P.off_btoo); }
  double* btil() const { return d(P.off_btil); }
  double* J() const { return d(P.off_J); }
  double* slabs() const { return d(P.off_slabs); }
  double* F() const { return d(P.off_F); }
  double* partial() const { return d(P.off_partial); }
  double* etrip() const { return d(P.off_etrip); }
  double* esum() const { return d(P.off_esum); }
  int* act_dev() const { return reinterpret_cast<int*>(ws + P.off_act); }
  int* orbits_dev() const { return reinterpret_cast<int*>(ws + P.off_orbits); }
  GemmTask* tasks_dev() const { return reinterpret_cast<GemmTask*>(ws + P.off_tasks); }
  TripletRec* trips_dev() const { return reinterpret_cast<TripletRec*>(ws + P.off_trips); }

  ~Ctx() {
    for (cudaEvent_t e : prof_main) cudaEventDestroy(e);
    for (cudaEvent_t e : prof_form) cudaEventDestroy(e);
    if (prof_begin) cudaEventDestroy(prof_begin);
    if (prof_prepared) cudaEventDestroy(prof_prepared);
    if (prof_end) cudaEventDestroy(prof_end);
    for (int s = 0; s < 4; ++s) {
      if (ev_formed[s]) cudaEventDestroy(ev_formed[s]);
      if (ev_free[s]) cudaEventDestroy(ev_free[s]);
    }
    if (ev_fork) cudaEventDestroy(ev_fork);
    if (ev_join) cudaEventDestroy(ev_join);
    if (s_form) cudaStreamDestroy(s_form);
    if (own_ws && ws) cudaFree(ws);
  }
};

struct Run { int pos0, orb0, len; };   // a run of consecutive orbitals inside the active list

std::vector<Run> runs_of(const std::vector<int>& act, int p0, int p1) {
  std::vector<Run> r;
  for (int p = p0; p < p1;) {
    int q = p + 1;
    while (q < p1 && act[q] == act[q - 1] + 1) ++q;
    r.push_back({p, act[p], q - p});
    p = q;
  }
  return r;
}

size_t push_task(Ctx& c, const GemmTask& t) {
  c.tasks.push_back(t);
  return c.tasks.size() - 1;
}

GemmTask single_term_task(long long c_off) {
  GemmTask t;
  memset(&t, 0, sizeof(t));
  t.nterms = 1;
  t.c_off = c_off;
  return t;
}

int tmap(CUtensorMap* m, const void* base, unsigned long long d0, unsigned long long d1, unsigned long long d2,
         unsigned long long d3, unsigned box1, unsigned box2) {
  const unsigned long long dims[4] = {d0, d1, d2, d3};
  const unsigned long long str[4] = {8, d0 * 8, d0 * d1 * 8, d0 * d1 * d2 * 8};
  return make_tensor_map_f64(m, base, dims, str, box1, box2);
}

// One strided-output DF GEMM: C = A[(m1,m2), Q] . B[n, Q]^T
struct DfGemm {
  const double* A; int a_d1, a_d2;          // A tensor [a_d2][a_d1][Xp]; rows (m1 in a_d2, m2 in a_d1)
  const double* B; long long b_rows;        // B tensor [b_rows][Xp]
  int m1_base, m1_ext, m2_ext;
  int n_base; long long n_ext;
  long long c_off, sM1, sM2, sN1, sN2; int n2_ext;
  double* C;
};

int run_df_gemm(Ctx& c, const DfGemm& g, size_t task_slot, cudaStream_t s) {
  const Plan& P = c.P;
  if (task_slot >= c.tasks.size() || c.tasks[task_slot].nterms != 1 || c.tasks[task_slot].c_off != g.c_off) {
    set_error(BQC_ERR_CUDA, "internal: DF task slot %zu does not match its launch", task_slot);
    return BQC_ERR_CUDA;
  }
  int tp, tql;
  choose_m_tile(g.m1_ext, g.m2_ext, &tp, &tql);
  const int tq = 1 << tql;
  const int nf = choose_nf(g.n_ext);
  CUtensorMap tA, tB;
  BQC_TRY(tmap(&tA, g.A, P.Xp, g.a_d1, g.a_d2, 1, tq, tp));
  BQC_TRY(tmap(&tB, g.B, P.Xp, g.b_rows, 1, 1, gemm_bn(nf), 1));
  GemmParams prm;
  memset(&prm, 0, sizeof(prm));
  prm.ntasks = 1;
  prm.tiles_m1 = ceil_div(g.m1_ext, tp);
  prm.tiles_m2 = ceil_div(g.m2_ext, tq);
  prm.tiles_n = (int)((g.n_ext + gemm_bn(nf) - 1) / gemm_bn(nf));
  prm.tp = tp; prm.tq_log2 = tql;
  prm.m1_base = g.m1_base; prm.n_base = g.n_base;
  prm.m1_ext = g.m1_ext; prm.m2_ext = g.m2_ext; prm.n_ext = (int)g.n_ext;
  prm.kiters = P.Xp / kBK;
  prm.out_mode = 0;
  prm.n2_ext = g.n2_ext;
  prm.sM1 = g.sM1; prm.sM2 = g.sM2; prm.sN1 = g.sN1; prm.sN2 = g.sN2;
  prm.tasks = c.tasks_dev() + task_slot;
  prm.C = g.C;
  return launch_gemm_nt(nf, tA, tA, tB, prm, s);
}

// ------------------------------------------------------------------ the pipeline
struct Action {
  enum Kind { FORM, COMPUTE } kind;
  int set, block;                 // FORM
  size_t trip0, ntrip, task0;     // COMPUTE (indices into the schedule arrays)
  int sets_used[3];
};

struct Pipeline {
  Ctx c;
  std::vector<Action> actions;
  std::vector<size_t> form_task_slot;   // per FORM action run: task slots (one per run)

  int setup(int o, int v, int X, const Inputs& in, const std::vector<int>& act, const bqc_t_opts* opts,
            void* workspace, size_t workspace_bytes, cudaStream_t stream);
  int prepare();                          // repack inputs, B~, J, zero-fills
  int form_block(int set, int block, cudaStream_t s);
  int build_schedule();
  int compute(const Action& a);
  int execute();
  int block_begin(int b) const { return b * c.P.Bo; }
  int block_end(int b) const { return std::min(c.P.na, (b + 1) * c.P.Bo); }
};

int Pipeline::setup(int o, int v, int X, const Inputs& in, const std::vector<int>& act,
                    const bqc_t_opts* opts, void* workspace, size_t workspace_bytes, cudaStream_t stream) {
  BQC_TRY(make_plan(c.P, o, v, X, act, opts));
  c.in = in;
  c.s_main = stream;
  if (workspace) {
    if (workspace_bytes < c.P.total || (reinterpret_cast<uintptr_t>(workspace) & 255)) {
      set_error(BQC_ERR_WORKSPACE, "workspace of %zu bytes (need %zu, 256-byte aligned)", workspace_bytes,
                c.P.total);
      return BQC_ERR_WORKSPACE;
    }
    c.ws = static_cast<uint8_t*>(workspace);
  } else {
    void* p = nullptr;
    cudaError_t e = cudaMalloc(&p, c.P.total);
    if (e != cudaSuccess) {
      cudaGetLastError();
      set_error(BQC_ERR_WORKSPACE, "cudaMalloc of %zu workspace bytes failed: %s", c.P.total,
                cudaGetErrorString(e));
      return BQC_ERR_WORKSPACE;
    }
    c.ws = static_cast<uint8_t*>(p);
    c.own_ws = true;
  }
  BQC_CUDA_OK(cudaStreamCreateWithFlags(&c.s_form, cudaStreamNonBlocking));
  for (int s = 0; s < 4; ++s) {
    BQC_CUDA_OK(cudaEventCreateWithFlags(&c.ev_formed[s], cudaEventDisableTiming));
    BQC_CUDA_OK(cudaEventCreateWithFlags(&c.ev_free[s], cudaEventDisableTiming));
  }
  BQC_CUDA_OK(cudaEventCreateWithFlags(&c.ev_fork, cudaEventDisableTiming));
  BQC_CUDA_OK(cudaEventCreateWithFlags(&c.ev_join, cudaEventDisableTiming));

  const Plan& P = c.P;
  c.f_nmseg = split_m(v, v, c.f_mseg);
  c.f_nseg = split_n(v, c.f_seg);
  for (int m = 0; m < c.f_nmseg; ++m) {
    const int tq = 1 << c.f_mseg[m].tq_log2;
    BQC_TRY(tmap(&c.tm_slab[m], c.slabs(), P.Kp, v, v, P.nslots, tq, c.f_mseg[m].tp));
    BQC_TRY(tmap(&c.tm_slabT[m], c.slabs(), P.Kp, v, v, P.nslots, 1, tq));
  }
  for (int n = 0; n < c.f_nseg; ++n)
    BQC_TRY(tmap(&c.tm_btil[n], c.btil(), P.Kp, v, (unsigned long long)P.na * P.na, 1, gemm_bn(c.f_seg[n].nf), 1));
  return BQC_OK;
}

// The W-builder GEMM of `prm.ntasks` tasks: one launch per (row segment, column segment).
int launch_f_gemm(Ctx& c, GemmParams prm, cudaStream_t s) {
  const int v = c.P.v;
  prm.m1_ext = v; prm.m2_ext = v; prm.n_ext = v;
  prm.kiters = c.P.Kp / kBK;
  prm.out_mode = 1;
  prm.nbv = c.P.nbv;
  prm.n2_ext = 1;
  for (int m = 0; m < c.f_nmseg; ++m) {
    const MSegment& ms = c.f_mseg[m];
    prm.tp = ms.tp; prm.tq_log2 = ms.tq_log2;
    prm.tiles_m1 = ms.tiles_m1;
    prm.tiles_m2 = ceil_div(v, 1 << ms.tq_log2);
    prm.m1_base = prm.m1_out = ms.m1_0;
    for (int n = 0; n < c.f_nseg; ++n) {
      prm.tiles_n = c.f_seg[n].ntiles;
      prm.n_base = prm.n_out = c.f_seg[n].n0;
      BQC_TRY(launch_gemm_nt(c.f_seg[n].nf, c.tm_slab[m], c.tm_slabT[m], c.tm_btil[n], prm, s));
    }
  }
  return BQC_OK;
}

int Pipeline::prepare() {
  const Plan& P = c.P;
  cudaStream_t s = c.s_main;
  const int o = P.o, v = P.v, X = P.X, na = P.na;
  // K-major copies of the DF factors: Bt[r][Q] = B[Q][r]
  BQC_TRY(launch_transpose_pad(c.in.B_vv, c.btvv(), X, v * v, P.Xp, s));
  BQC_TRY(launch_transpose_pad(c.in.B_ov, c.btov(), X, o * v, P.Xp, s));
  BQC_TRY(launch_transpose_pad(c.in.B_oo, c.btoo(), X, o * o, P.Xp, s));
  // zero fills: K padding of B~ and slabs, pad blocks of F, per-triplet energies
  BQC_CUDA_OK(cudaMemsetAsync(c.btil(), 0, (size_t)na * na * v * P.Kp * 8, s));
  BQC_CUDA_OK(cudaMemsetAsync(c.slabs(), 0, (size_t)P.nslots * P.slab_elems * 8, s));
  BQC_CUDA_OK(cudaMemsetAsync(c.F(), 0, (size_t)P.nbatch * 3 * P.fsz * 8, s));
  BQC_CUDA_OK(cudaMemsetAsync(c.etrip(), 0, num_triplets(o) * 8, s));
  BQC_CUDA_OK(cudaMemcpyAsync(c.act_dev(), P.act.data(), (size_t)na * 4, cudaMemcpyHostToDevice, s));
  // orbit table A <= B <= C
  {
    std::vector<int> orb;
    orb.reserve(P.norbits);
    for (int A = 0; A < P.nbv; ++A)
      for (int B = A; B < P.nbv; ++B)
        for (int C = B; C < P.nbv; ++C) orb.push_back(A | (B << 10) | (C << 20));
    BQC_CUDA_OK(cudaMemcpyAsync(c.orbits_dev(), orb.data(), orb.size() * 4, cudaMemcpyHostToDevice, s));
    BQC_CUDA_OK(cudaStreamSynchronize(s));   // `orb` goes out of scope
  }
  // the whole schedule (GEMM tasks + triplet records) goes up once
  if (c.tasks.size() > P.max_tasks || c.trips.size() > P.max_trips) {
    set_error(BQC_ERR_WORKSPACE, "internal: schedule arrays overflow (%zu/%zu tasks, %zu/%zu triplets)",
              c.tasks.size(), P.max_tasks, c.trips.size(), P.max_trips);
    return BQC_ERR_WORKSPACE;
  }
  if (!c.tasks.empty())
    BQC_CUDA_OK(cudaMemcpyAsync(c.tasks_dev(), c.tasks.data(), c.tasks.size() * sizeof(GemmTask),
                                cudaMemcpyHostToDevice, s));
  if (!c.trips.empty())
    BQC_CUDA_OK(cudaMemcpyAsync(c.trips_dev(), c.trips.data(), c.trips.size() * sizeof(TripletRec),
                                cudaMemcpyHostToDevice, s));

  // B~ particle columns: t2 rows
  BQC_TRY(launch_btilde_t2(c.in.t2, c.btil(), o, v, c.act_dev(), na, P.Kp, s));
  // B~ hole columns (z r|y l) and J_xy[u,w] = (x u|y w), one GEMM per pair of contiguous runs
  const std::vector<Run> runs = runs_of(P.act, 0, na);
  size_t slot = 0;   // DF tasks occupy the first slots of the task array (see build_schedule)
  for (const Run& rz : runs)
    for (const Run& ry : runs) {
      DfGemm g;
      g.A = c.btov(); g.a_d1 = v; g.a_d2 = o;
      g.B = c.btoo(); g.b_rows = (long long)o * o;
      g.m1_base = rz.orb0; g.m1_ext = rz.len; g.m2_ext = v;
      g.n_base = ry.orb0 * o; g.n_ext = (long long)ry.len * o;
      g.c_off = ((long long)rz.pos0 * na + ry.pos0) * v * P.Kp + v;
      g.sM1 = (long long)na * v * P.Kp; g.sM2 = P.Kp; g.sN1 = (long long)v * P.Kp; g.sN2 = 1; g.n2_ext = o;
      g.C = c.btil();
      BQC_TRY(run_df_gemm(c, g, slot++, s));
      DfGemm j;
      j.A = c.btov(); j.a_d1 = v; j.a_d2 = o;
      j.B = c.btov(); j.b_rows = (long long)o * v;
      j.m1_base = rz.orb0; j.m1_ext = rz.len; j.m2_ext = v;
      j.n_base = ry.orb0 * v; j.n_ext = (long long)ry.len * v;
      j.c_off = ((long long)rz.pos0 * na + ry.pos0) * v * v;
      j.sM1 = (long long)na * v * v; j.sM2 = v; j.sN1 = (long long)v * v; j.sN2 = 1; j.n2_ext = v;
      j.C = c.J();
      BQC_TRY(run_df_gemm(c, j, slot++, s));
    }
  // the former stream starts after the repacked inputs exist
  BQC_CUDA_OK(cudaEventRecord(c.ev_fork, s));
  BQC_CUDA_OK(cudaStreamWaitEvent(c.s_form, c.ev_fork, 0));
  return BQC_OK;
}

// Augmented slabs of one occupied block into slot set `set` (row a1 + hole columns).
int Pipeline::form_block(int set, int block, cudaStream_t s) {
  const Plan& P = c.P;
  const int v = P.v;
  const int p0 = block_begin(block), p1 = block_end(block);
  for (const Run& r : runs_of(P.act, p0, p1)) {
    const int slot0 = set * P.Bo + (r.pos0 - p0);
    DfGemm g;
    g.A = c.btvv(); g.a_d1 = v; g.a_d2 = v;             // rows (m1 = q, m2 = d)
    g.B = c.btov(); g.b_rows = (long long)P.o * v;      // rows n = (x, p)
    g.m1_base = 0; g.m1_ext = v; g.m2_ext = v;
    g.n_base = r.orb0 * v; g.n_ext = (long long)r.len * v;
    g.c_off = (long long)slot0 * (long long)P.slab_elems;
    g.sM1 = P.Kp; g.sM2 = 1; g.sN1 = 0; g.sN2 = (long long)v * P.Kp; g.n2_ext = INT_MAX;
    g.C = c.slabs();
    // DF tasks are all "single term, a_idx = b_idx = 0" and differ only in c_off; slot reserved in build_schedule
    BQC_TRY(run_df_gemm(c, g, form_task_slot[(size_t)block * P.nsets * P.na + (size_t)set * P.na + r.pos0], s));
    BQC_TRY(launch_slab_holes(c.in.t2, c.slabs(), P.o, v, P.Kp, r.orb0, r.len, slot0, s));
  }
  return BQC_OK;
}

int Pipeline::build_schedule() {
  Plan& P = c.P;
  const int na = P.na, v = P.v;
  // ---- DF task slots first: (z-run, y-run) pairs for B~/J, then one per (block, set, run) for slabs
  const std::vector<Run> runs = runs_of(P.act, 0, na);
  for (const Run& rz : runs)
    for (const Run& ry : runs) {
      push_task(c, single_term_task(((long long)rz.pos0 * na + ry.pos0) * v * P.Kp + v));
      push_task(c, single_term_task(((long long)rz.pos0 * na + ry.pos0) * v * v));
    }
  form_task_slot.assign((size_t)P.nblk * P.nsets * na, (size_t)-1);
  for (int b = 0; b < P.nblk; ++b)
    for (int set = 0; set < P.nsets; ++set)
      for (const Run& r : runs_of(P.act, block_begin(b), block_end(b))) {
        const int slot0 = set * P.Bo + (r.pos0 - block_begin(b));
        form_task_slot[(size_t)b * P.nsets * na + (size_t)set * na + r.pos0] =
            push_task(c, single_term_task((long long)slot0 * (long long)P.slab_elems));
      }

  // ---- block triples I <= J <= K with the slot-set protocol: I -> set 0, J -> set 1, K -> sets 2/3
  int set_block[4] = {-1, -1, -1, -1};
  int kflip = 0;
  auto acquire = [&](int set, int block) {
    if (set_block[set] == block) return;
    Action a;
    memset(&a, 0, sizeof(a));
    a.kind = Action::FORM; a.set = set; a.block = block;
    actions.push_back(a);
    set_block[set] = block;
  };
  auto slot_of = [&](int pos, int set, int block) { return set * P.Bo + (pos - block_begin(block)); };

  long long block_triple = -1;
  std::vector<int> bt_owner;
  if (P.shard_blocks) bt_owner = deal_block_triples(na, P.Bo, P.shard_count);
  for (int I = 0; I < P.nblk; ++I) {
    for (int Jb = I; Jb < P.nblk; ++Jb) {
      const int sJ = (Jb == I) ? 0 : 1;
      for (int K = Jb; K < P.nblk; ++K) {
        ++block_triple;
        // BQC_T_FLAG_SHARD_BLOCKS: whole block triples are dealt to the shards, so a shard forms only the
        // slabs of its own block triples; otherwise every shard owns some triplets of every block triple
        if (P.shard_blocks && bt_owner[(size_t)block_triple] != P.shard_rank) continue;
        int sK = sJ;
        if (K != Jb) sK = (set_block[2] == K) ? 2 : (set_block[3] == K ? 3 : 2 + (kflip++ & 1));
        // triplets of this block triple owned by this shard
        std::vector<TripletRec> list;
        std::vector<int> slots;   // 3 per triplet
        for (int pi = block_begin(I); pi < block_end(I); ++pi)
          for (int pj = std::max(pi, block_begin(Jb)); pj < block_end(Jb); ++pj)
            for (int pk = std::max(pj, block_begin(K)); pk < block_end(K); ++pk) {
              if (pi == pj && pj == pk) continue;   // g(i,i,i) = 0 exactly
              TripletRec t;
              t.i = P.act[pi]; t.j = P.act[pj]; t.k = P.act[pk];
              t.pi = pi; t.pj = pj; t.pk = pk;
              t.index = (long long)triplet_index(P.o, t.i, t.j, t.k);
              if (!P.shard_blocks && (int)(t.index % P.shard_count) != P.shard_rank) continue;
              list.push_back(t);
              slots.push_back(slot_of(pi, 0, I));
              slots.push_back(slot_of(pj, sJ, Jb));
              slots.push_back(slot_of(pk, sK, K));
            }
        if (list.empty()) continue;
        // slabs are formed only for block triples that have work (the acquire calls are idempotent)
        acquire(0, I);
        if (Jb != I) acquire(1, Jb);
        if (K != Jb) acquire(sK, K);
        for (size_t b0 = 0; b0 < list.size(); b0 += P.nbatch) {
          const size_t nb = std::min(list.size() - b0, (size_t)P.nbatch);
          Action a;
          memset(&a, 0, sizeof(a));
          a.kind = Action::COMPUTE;
          a.trip0 = c.trips.size(); a.ntrip = nb; a.task0 = c.tasks.size();
          a.sets_used[0] = 0; a.sets_used[1] = sJ; a.sets_used[2] = sK;
          for (size_t n = 0; n < nb; ++n) {
            const TripletRec& t = list[b0 + n];
            const int si = slots[3 * (b0 + n)], sj = slots[3 * (b0 + n) + 1], sk = slots[3 * (b0 + n) + 2];
            c.trips.push_back(t);
            auto pair = [&](int pz, int py) { return pz * na + py; };
            // F(x,y,z): term0 = (I~_x, canonical rows, B~_zy), term1 = (I~_y, transposed rows, B~_zx)
            auto f_task = [&](int sx, int sy, int px, int py, int pz, int cls) {
              GemmTask g;
              memset(&g, 0, sizeof(g));
              g.nterms = 2;
              g.term[0].a_idx = sx; g.term[0].a_transposed = 0; g.term[0].b_idx = pair(pz, py);
              g.term[1].a_idx = sy; g.term[1].a_transposed = 1; g.term[1].b_idx = pair(pz, px);
              g.c_off = (long long)((n * 3 + cls) * P.fsz);
              push_task(c, g);
            };
            f_task(si, sj, t.pi, t.pj, t.pk, 0);   // F(i,j,k)
            f_task(si, sk, t.pi, t.pk, t.pj, 1);   // F(i,k,j)
            f_task(sj, sk, t.pj, t.pk, t.pi, 2);   // F(j,k,i)
          }
          actions.push_back(a);
        }
      }
    }
  }
  return BQC_OK;
}

int Pipeline::compute(const Action& a) {
  const Plan& P = c.P;
  cudaStream_t s = c.s_main;
  const int v = P.v;
  GemmParams prm;
  memset(&prm, 0, sizeof(prm));
  prm.ntasks = (int)(3 * a.ntrip);
  prm.tasks = c.tasks_dev() + a.task0;
  prm.C = c.F();
  if (P.profile) BQC_TRY(c.prof_mark(c.prof_main, s));
  BQC_TRY(launch_f_gemm(c, prm, s));
  if (P.profile) BQC_TRY(c.prof_mark(c.prof_main, s));

  EnergyArgs e;
  e.F = c.F(); e.trips = c.trips_dev() + a.trip0; e.orbits = c.orbits_dev();
  e.J = c.J(); e.t1 = c.in.t1; e.eps_occ = c.in.eps_occ; e.eps_vir = c.in.eps_vir;
  e.partial = c.partial();
  e.t2 = c.in.t2; e.f_ov = c.in.f_ov; e.o = P.o;
  e.ntrip = (int)a.ntrip; e.norbits = P.norbits; e.nbv = P.nbv; e.v = v; e.nw = P.na; e.use_t1 = P.use_t1;
  BQC_TRY(launch_energy(e, s));
  BQC_TRY(launch_reduce_triplets(c.partial(), c.trips_dev() + a.trip0, (int)a.ntrip, P.norbits, c.etrip(), s));
  if (P.profile) BQC_TRY(c.prof_mark(c.prof_main, s));
  return BQC_OK;
}

int Pipeline::execute() {
  for (const Action& a : actions) {
    if (a.kind == Action::FORM) {
      // the former stream may overwrite a slot set only after the main stream's last use of it
      if (c.ev_free_valid[a.set]) BQC_CUDA_OK(cudaStreamWaitEvent(c.s_form, c.ev_free[a.set], 0));
      if (c.P.profile) BQC_TRY(c.prof_mark(c.prof_form, c.s_form));
      BQC_TRY(form_block(a.set, a.block, c.s_form));
      if (c.P.profile) BQC_TRY(c.prof_mark(c.prof_form, c.s_form));
      BQC_CUDA_OK(cudaEventRecord(c.ev_formed[a.set], c.s_form));
      BQC_CUDA_OK(cudaStreamWaitEvent(c.s_main, c.ev_formed[a.set], 0));
    } else {
      BQC_TRY(compute(a));
      for (int n = 0; n < 3; ++n) {
        const int set = a.sets_used[n];
        BQC_CUDA_OK(cudaEventRecord(c.ev_free[set], c.s_main));
        c.ev_free_valid[set] = true;
      }
    }
  }
  // join the former stream back into the caller's stream
  BQC_CUDA_OK(cudaEventRecord(c.ev_join, c.s_form));
  BQC_CUDA_OK(cudaStreamWaitEvent(c.s_main, c.ev_join, 0));
  return BQC_OK;
}

// ------------------------------------------------------------------ common front end
int validate_inputs(int o, int v, int X, const Inputs& in) {
  BQC_TRY(check_sizes(o, v, X));
  BQC_TRY(check_device());
  BQC_TRY(check_device_ptr(in.eps_occ, "eps_occ"));
  BQC_TRY(check_device_ptr(in.eps_vir, "eps_vir"));
  BQC_TRY(check_device_ptr(in.t1, "t1"));
  BQC_TRY(check_device_ptr(in.t2, "t2"));
  BQC_TRY(check_device_ptr(in.B_oo, "B_oo"));
  BQC_TRY(check_device_ptr(in.B_ov, "B_ov"));
  BQC_TRY(check_device_ptr(in.B_vv, "B_vv"));
  return BQC_OK;
}

int check_denominators(int o, int v, const Inputs& in, cudaStream_t s) {
  std::vector<double> eo(o), ev(v);
  BQC_CUDA_OK(cudaMemcpyAsync(eo.data(), in.eps_occ, (size_t)o * 8, cudaMemcpyDeviceToHost, s));
  BQC_CUDA_OK(cudaMemcpyAsync(ev.data(), in.eps_vir, (size_t)v * 8, cudaMemcpyDeviceToHost, s));
  BQC_CUDA_OK(cudaStreamSynchronize(s));
  const double emax = *std::max_element(eo.begin(), eo.end());
  const double vmin = *std::min_element(ev.begin(), ev.end());
  if (!(3.0 * emax - 3.0 * vmin < 0.0)) {
    set_error(BQC_ERR_DENOMINATOR, "3*max(eps_occ)=%g - 3*min(eps_vir)=%g >= 0: denominators may vanish",
              3.0 * emax, 3.0 * vmin);
    return BQC_ERR_DENOMINATOR;
  }
  return BQC_OK;
}

int t_energy_impl(int o, int v, int X, const Inputs& in, const bqc_t_opts* opts, void* workspace,
                  size_t workspace_bytes, double* e_total_host, double* e_triplet_dev, cudaStream_t stream) {
  clear_error();
  if (!e_total_host) {
    set_error(BQC_ERR_NULL_POINTER, "e_total_host is NULL");
    return BQC_ERR_NULL_POINTER;
  }
  BQC_TRY(validate_inputs(o, v, X, in));
  if (in.f_ov) BQC_TRY(check_device_ptr(in.f_ov, "opts->f_ov"));
  if (e_triplet_dev) BQC_TRY(check_device_ptr(e_triplet_dev, "e_triplet_dev"));
  int lo, hi;
  BQC_TRY(resolve_window(o, opts, &lo, &hi));
  BQC_TRY(check_denominators(o, v, in, stream));
  if (hi - lo < 2) {   // a single occupied orbital: two electrons, no triples
    *e_total_host = 0.0;
    if (e_triplet_dev) BQC_CUDA_OK(cudaMemsetAsync(e_triplet_dev, 0, num_triplets(o) * 8, stream));
    BQC_CUDA_OK(cudaStreamSynchronize(stream));
    return BQC_OK;
  }
  std::vector<int> act;
  for (int x = lo; x < hi; ++x) act.push_back(x);

  Pipeline p;
  BQC_TRY(p.setup(o, v, X, in, act, opts, workspace, workspace_bytes, stream));
  Ctx& c = p.c;
  const bool prof = c.P.profile != 0;
  const long long launches0 = g_launches;
  if (prof) {
    BQC_CUDA_OK(cudaEventCreate(&c.prof_begin));
    BQC_CUDA_OK(cudaEventCreate(&c.prof_prepared));
    BQC_CUDA_OK(cudaEventCreate(&c.prof_end));
    BQC_CUDA_OK(cudaEventRecord(c.prof_begin, stream));
  }
  BQC_TRY(p.build_schedule());
  BQC_TRY(p.prepare());
  if (prof) BQC_CUDA_OK(cudaEventRecord(c.prof_prepared, stream));
  BQC_TRY(p.execute());
  BQC_TRY(launch_final_sum(c.etrip(), (long long)num_triplets(o), c.esum(), stream));
  if (prof) BQC_CUDA_OK(cudaEventRecord(c.prof_end, stream));
  if (e_triplet_dev)
    BQC_CUDA_OK(cudaMemcpyAsync(e_triplet_dev, c.etrip(), num_triplets(o) * 8, cudaMemcpyDeviceToDevice, stream));
  BQC_CUDA_OK(cudaMemcpyAsync(e_total_host, c.esum(), 8, cudaMemcpyDeviceToHost, stream));
  BQC_CUDA_OK(cudaStreamSynchronize(stream));
  BQC_CUDA_OK(cudaStreamSynchronize(c.s_form));
  g_profile[8] = (double)(g_launches - launches0);
  if (prof) {
    double gemm_ms = 0, en_ms = 0, form_ms = 0;
    float ms = 0.f;
    for (size_t n = 0; n + 2 < c.prof_main.size() + 1; n += 3) {
      BQC_CUDA_OK(cudaEventElapsedTime(&ms, c.prof_main[n], c.prof_main[n + 1]));
      gemm_ms += ms;
      BQC_CUDA_OK(cudaEventElapsedTime(&ms, c.prof_main[n + 1], c.prof_main[n + 2]));
      en_ms += ms;
    }
    for (size_t n = 0; n + 1 < c.prof_form.size(); n += 2) {
      BQC_CUDA_OK(cudaEventElapsedTime(&ms, c.prof_form[n], c.prof_form[n + 1]));
      form_ms += ms;
    }
    g_profile[0] = gemm_ms;
    g_profile[1] = (double)(c.prof_main.size() / 3);
    g_profile[2] = en_ms;
    g_profile[3] = (double)(c.prof_main.size() / 3);
    g_profile[4] = form_ms;
    g_profile[5] = (double)(c.prof_form.size() / 2);
    BQC_CUDA_OK(cudaEventElapsedTime(&ms, c.prof_begin, c.prof_prepared));
    g_profile[6] = ms;
    BQC_CUDA_OK(cudaEventElapsedTime(&ms, c.prof_begin, c.prof_end));
    g_profile[7] = ms;
  }
  return BQC_OK;
}

// ------------------------------------------------------------------ abc-driven schedule
// The paper's loop is over virtual triples a,b,c with o^3 tensors per iteration.  The
// contraction of Eq. (2) is invariant under exchanging the roles of occupied and virtual orbitals
// (DESIGN.md §12): with
//     o' = v, v' = o, eps_occ' = -eps_vir, eps_vir' = -eps_occ, t1'[a,i] = t1[i,a],
//     t2'[a,b,i,j] = -t2[i,j,a,b], B_oo' = B_vv, B_vv' = B_oo, B_ov'[Q,a,i] = B_ov[Q,i,a], f'[a,i] = -f[i,a]
// the dual problem's triplet (a <= b <= c) carries W_abc[i,j,k] for all i,j,k, its "slabs" are the o^2 (v+o)
// pieces (zr|yl), t2[z,y,r,:] of one virtual r and its per-triplet value is the abc-driven contribution
// (2 - d_ab - d_bc) sum_ijk R V / D.  So the abc-driven schedule is the same pipeline on the dual arrays,
// which are built here on the device (one pass over t2 and B_ov).
struct DualLayout {
  size_t off_eo = 0, off_ev = 0, off_t1 = 0, off_f = 0, off_bov = 0, off_t2 = 0, total = 0;
};

DualLayout dual_layout(int o, int v, int X, bool fock) {
  DualLayout L;
  size_t off = 0;
  auto take = [&](size_t bytes) { size_t r = off; off = round_up(off + bytes, 1024); return r; };
  L.off_eo = take((size_t)v * 8);
  L.off_ev = take((size_t)o * 8);
  L.off_t1 = take((size_t)o * v * 8);
  L.off_f = take(fock ? (size_t)o * v * 8 : 0);
  L.off_bov = take((size_t)X * o * v * 8);
  L.off_t2 = take((size_t)o * o * v * v * 8);
  L.total = off;
  return L;
}

bqc_t_opts dual_opts(const bqc_t_opts* opts) {
  bqc_t_opts d;
  memset(&d, 0, sizeof(d));
  if (opts) d = *opts;
  d.flags &= ~BQC_T_FLAG_ABC_DRIVEN;
  d.f_ov = nullptr;
  return d;
}

int t_energy_abc(int o, int v, int X, const Inputs& in, const bqc_t_opts* opts, void* workspace,
                 size_t workspace_bytes, double* e_total_host, double* e_triplet_dev, cudaStream_t stream) {
  clear_error();
  if (!e_total_host) {
    set_error(BQC_ERR_NULL_POINTER, "e_total_host is NULL");
    return BQC_ERR_NULL_POINTER;
  }
  BQC_TRY(validate_inputs(o, v, X, in));
  if (in.f_ov) BQC_TRY(check_device_ptr(in.f_ov, "opts->f_ov"));
  bqc_t_opts dopts = dual_opts(opts);
  int lo, hi;
  BQC_TRY(resolve_window(v, &dopts, &lo, &hi));
  Plan P;
  {
    std::vector<int> act(hi - lo);
    for (int x = lo; x < hi; ++x) act[x - lo] = x;
    BQC_TRY(make_plan(P, v, o, X, act, &dopts));
  }
  const DualLayout L = dual_layout(o, v, X, in.f_ov != nullptr);
  const size_t need = L.total + P.total;
  uint8_t* ws = static_cast<uint8_t*>(workspace);
  bool own = false;
  if (ws) {
    if (workspace_bytes < need || (reinterpret_cast<uintptr_t>(ws) & 255)) {
      set_error(BQC_ERR_WORKSPACE, "workspace of %zu bytes (need %zu, 256-byte aligned)", workspace_bytes, need);
      return BQC_ERR_WORKSPACE;
    }
  } else {
    void* p = nullptr;
    cudaError_t e = cudaMalloc(&p, need);
    if (e != cudaSuccess) {
      cudaGetLastError();
      set_error(BQC_ERR_WORKSPACE, "cudaMalloc of %zu workspace bytes failed: %s", need, cudaGetErrorString(e));
      return BQC_ERR_WORKSPACE;
    }
    ws = static_cast<uint8_t*>(p);
    own = true;
  }
  auto D = [&](size_t off) { return reinterpret_cast<double*>(ws + off); };
  const long long launches0 = g_launches;
  int rc = launch_transpose_scale(in.eps_vir, D(L.off_eo), 1, 1, v, -1.0, stream);
  if (rc == BQC_OK) rc = launch_transpose_scale(in.eps_occ, D(L.off_ev), 1, 1, o, -1.0, stream);
  if (rc == BQC_OK) rc = launch_transpose_scale(in.t1, D(L.off_t1), 1, o, v, 1.0, stream);
  if (rc == BQC_OK && in.f_ov) rc = launch_transpose_scale(in.f_ov, D(L.off_f), 1, o, v, -1.0, stream);
  if (rc == BQC_OK) rc = launch_transpose_scale(in.B_ov, D(L.off_bov), X, o, v, 1.0, stream);
  if (rc == BQC_OK)
    rc = launch_transpose_scale(in.t2, D(L.off_t2), 1, (long long)o * o, (long long)v * v, -1.0, stream);
  if (rc == BQC_OK) {
    Inputs din = {D(L.off_eo), D(L.off_ev), D(L.off_t1), D(L.off_t2), in.B_vv, D(L.off_bov), in.B_oo,
                  in.f_ov ? D(L.off_f) : nullptr};
    rc = t_energy_impl(v, o, X, din, &dopts, ws + L.total, P.total, e_total_host, e_triplet_dev, stream);
    g_profile[8] = (double)(g_launches - launches0);
  }
  if (own) {
    cudaStreamSynchronize(stream);
    cudaFree(ws);
  }
  return rc;
}

}  // namespace
}  // namespace bqc

// ====================================================================== C ABI
using namespace bqc;

extern "C" {

size_t bqc_t_num_triplets(int nocc) { return nocc > 0 ? num_triplets(nocc) : 0; }

size_t bqc_t_triplet_index(int nocc, int i, int j, int k) {
  if (nocc <= 0 || i < 0 || i > j || j > k || k >= nocc) return (size_t)-1;
  return triplet_index(nocc, i, j, k);
}

int bqc_t_triplet_owner(int nocc, int shard_count, int i, int j, int k) {
  const size_t idx = bqc_t_triplet_index(nocc, i, j, k);
  if (idx == (size_t)-1 || shard_count <= 0) return -1;
  return (int)(idx % (size_t)shard_count);
}

int bqc_t_triplet_owner_ex(int nocc, int nvir, int naux, const bqc_t_opts* opts, int i, int j, int k) {
  clear_error();
  if (check_sizes(nocc, nvir, naux) != BQC_OK) return -1;
  if (opts && (opts->flags & BQC_T_FLAG_ABC_DRIVEN)) {   // (i,j,k) are virtual indices a<=b<=c
    const bqc_t_opts d = dual_opts(opts);
    return bqc_t_triplet_owner_ex(nvir, nocc, naux, &d, i, j, k);
  }
  int lo, hi;
  if (resolve_window(nocc, opts, &lo, &hi) != BQC_OK) return -1;
  if (i < lo || i > j || j > k || k >= hi) return -1;
  const int sc = (opts && opts->shard_count > 0) ? opts->shard_count : 1;
  if (!(opts && (opts->flags & BQC_T_FLAG_SHARD_BLOCKS)))
    return (int)(triplet_index(nocc, i, j, k) % (size_t)sc);
  Plan P;
  std::vector<int> act(hi - lo);
  for (int x = lo; x < hi; ++x) act[x - lo] = x;
  bqc_t_opts o2 = *opts;
  o2.shard_rank = 0;
  if (make_plan(P, nocc, nvir, naux, act, &o2) != BQC_OK) return -1;
  // block triples I <= J <= K are numbered in loop order = lexicographic rank among the nblk blocks
  const size_t bt = triplet_index(P.nblk, (i - lo) / P.Bo, (j - lo) / P.Bo, (k - lo) / P.Bo);
  return deal_block_triples(P.na, P.Bo, sc)[bt];
}

double bqc_t_flops(int nocc, int nvir, const bqc_t_opts* opts) {
  clear_error();
  if (nocc <= 0 || nvir <= 0) return 0.0;
  if (opts && (opts->flags & BQC_T_FLAG_ABC_DRIVEN)) {   // virtual triples a<=b<=c, 12 o^3 (v+o) each
    const bqc_t_opts d = dual_opts(opts);
    return bqc_t_flops(nvir, nocc, &d);
  }
  int lo, hi;
  if (resolve_window(nocc, opts, &lo, &hi) != BQC_OK) return -1.0;
  const int sc = (opts && opts->shard_count > 0) ? opts->shard_count : 1;
  const int sr = opts ? opts->shard_rank : 0;
  size_t n = 0;
  if (opts && (opts->flags & BQC_T_FLAG_SHARD_BLOCKS) && sc > 1) {
    // same block-triple walk as Pipeline::build_schedule (the block size does not depend on naux)
    Plan P;
    std::vector<int> act(hi - lo);
    for (int x = lo; x < hi; ++x) act[x - lo] = x;
    if (make_plan(P, nocc, nvir, 1, act, opts) != BQC_OK) return -1.0;
    std::vector<long long> load;
    deal_block_triples(P.na, P.Bo, sc, &load);
    n = (size_t)load[sr];
    const double v = nvir;
    return (double)n * 12.0 * v * v * v * (v + nocc);
  }
  for (int i = lo; i < hi; ++i)
    for (int j = i; j < hi; ++j)
      for (int k = j; k < hi; ++k) {
        if (i == j && j == k) continue;
        if ((int)(triplet_index(nocc, i, j, k) % (size_t)sc) == sr) ++n;
      }
  const double v = nvir;
  return (double)n * 12.0 * v * v * v * (v + nocc);
}

int bqc_t_plan_occ_block(int nocc, int nvir, int naux, const bqc_t_opts* opts) {
  clear_error();
  if (check_sizes(nocc, nvir, naux) != BQC_OK) return -1;
  if (opts && (opts->flags & BQC_T_FLAG_ABC_DRIVEN)) {   // block size over the virtual index
    const bqc_t_opts d = dual_opts(opts);
    return bqc_t_plan_occ_block(nvir, nocc, naux, &d);
  }
  int lo, hi;
  if (resolve_window(nocc, opts, &lo, &hi) != BQC_OK) return -1;
  Plan P;
  std::vector<int> act(hi - lo);
  for (int x = lo; x < hi; ++x) act[x - lo] = x;
  if (make_plan(P, nocc, nvir, naux, act, opts) != BQC_OK) return -1;
  return P.Bo;
}

size_t bqc_t_workspace_bytes(int nocc, int nvir, int naux, const bqc_t_opts* opts) {
  clear_error();
  if (check_sizes(nocc, nvir, naux) != BQC_OK) return 0;
  if (opts && (opts->flags & BQC_T_FLAG_ABC_DRIVEN)) {   // dual arrays + the dual problem's workspace
    const bqc_t_opts d = dual_opts(opts);
    const size_t inner = bqc_t_workspace_bytes(nvir, nocc, naux, &d);
    return inner ? dual_layout(nocc, nvir, naux, opts->f_ov != nullptr).total + inner : 0;
  }
  int lo, hi;
  if (resolve_window(nocc, opts, &lo, &hi) != BQC_OK) return 0;
  Plan P;
  std::vector<int> act(hi - lo);
  for (int x = lo; x < hi; ++x) act[x - lo] = x;
  if (make_plan(P, nocc, nvir, naux, act, opts) != BQC_OK) return 0;
  return P.total;
}

int bqc_sum_in_order(const double* x, size_t n, double* out_host, void* stream_v) {
  clear_error();
  if (!out_host || (!x && n > 0)) {
    set_error(BQC_ERR_NULL_POINTER, "bqc_sum_in_order: %s is NULL", out_host ? "x" : "out_host");
    return BQC_ERR_NULL_POINTER;
  }
  if (n == 0) {
    *out_host = 0.0;
    return BQC_OK;
  }
  cudaPointerAttributes attr;
  const cudaError_t e = cudaPointerGetAttributes(&attr, x);
  if (e != cudaSuccess) cudaGetLastError();   // no driver / no device: x can only be host memory
  if (e == cudaSuccess && (attr.type == cudaMemoryTypeDevice || attr.type == cudaMemoryTypeManaged)) {
    cudaStream_t stream = static_cast<cudaStream_t>(stream_v);
    double* d = nullptr;
    BQC_CUDA_OK(cudaMallocAsync(&d, 8, stream));
    int rc = launch_ordered_sum(x, (long long)n, d, stream);
    if (rc == BQC_OK) {
      cudaError_t c = cudaMemcpyAsync(out_host, d, 8, cudaMemcpyDeviceToHost, stream);
      if (c == cudaSuccess) c = cudaStreamSynchronize(stream);
      if (c != cudaSuccess) {
        set_error(BQC_ERR_CUDA, "bqc_sum_in_order: %s", cudaGetErrorString(c));
        rc = BQC_ERR_CUDA;
      }
    }
    cudaFreeAsync(d, stream);
    return rc;
  }
  double s = 0.0;
  for (size_t i = 0; i < n; ++i) s += x[i];   // the same left-to-right order as ordered_sum_kernel
  *out_host = s;
  return BQC_OK;
}

int bqc_t_last_profile(double* out, int n) {
  if (!out || n <= 0) return 0;
  const int m = n < 9 ? n : 9;
  for (int i = 0; i < m; ++i) out[i] = g_profile[i];
  return m;
}

int bqc_last_error(void) { return g_err; }
const char* bqc_error_detail(void) { return g_detail; }
const char* bqc_version(void) { return "bqc_t 0.1 (sm_100a)"; }

const char* bqc_error_string(int code) {
  switch (code) {
    case BQC_OK: return "ok";
    case BQC_ERR_INVALID_SIZE: return "invalid size";
    case BQC_ERR_NULL_POINTER: return "null pointer";
    case BQC_ERR_NOT_DEVICE_PTR: return "pointer is not in the expected memory space";
    case BQC_ERR_MISALIGNED: return "pointer is not 8-byte aligned";
    case BQC_ERR_WORKSPACE: return "workspace too small or allocation failed";
    case BQC_ERR_CUDA: return "CUDA error";
    case BQC_ERR_DEVICE: return "device is not sm_100 (B200)";
    case BQC_ERR_DENOMINATOR: return "non-negative orbital-energy denominator possible";
    case BQC_ERR_INVALID_OPTION: return "invalid option";
  }
  return "unknown error";
}

int bqc_t_energy_ex(int nocc, int nvir, int naux, const double* eps_occ, const double* eps_vir,
                    const double* t1, const double* t2, const double* B_oo, const double* B_ov,
                    const double* B_vv, const bqc_t_opts* opts, void* workspace, size_t workspace_bytes,
                    double* e_total_host, double* e_triplet_dev, void* stream) {
  Inputs in = {eps_occ, eps_vir, t1, t2, B_oo, B_ov, B_vv, opts ? opts->f_ov : nullptr};
  if (opts && (opts->flags & BQC_T_FLAG_ABC_DRIVEN))
    return t_energy_abc(nocc, nvir, naux, in, opts, workspace, workspace_bytes, e_total_host, e_triplet_dev,
                        static_cast<cudaStream_t>(stream));
  return t_energy_impl(nocc, nvir, naux, in, opts, workspace, workspace_bytes, e_total_host, e_triplet_dev,
                       static_cast<cudaStream_t>(stream));
}

double bqc_t_energy(int nocc, int nvir, int naux, const double* eps_occ, const double* eps_vir,
                    const double* t1, const double* t2, const double* B_oo, const double* B_ov,
                    const double* B_vv, void* stream) {
  double e = 0.0;
  const int rc = bqc_t_energy_ex(nocc, nvir, naux, eps_occ, eps_vir, t1, t2, B_oo, B_ov, B_vv, nullptr, nullptr,
                                 0, &e, nullptr, stream);
  return rc == BQC_OK ? e : nan("");
}

int bqc_t_energy_host(int nocc, int nvir, int naux, const double* eps_occ, const double* eps_vir,
                      const double* t1, const double* t2, const double* B_oo, const double* B_ov,
                      const double* B_vv, const bqc_t_opts* opts, double* e_total_host,
                      double* e_triplet_host, size_t* h2d_bytes, size_t* d2h_bytes, void* stream_v) {
  clear_error();
  cudaStream_t stream = static_cast<cudaStream_t>(stream_v);
  BQC_TRY(check_sizes(nocc, nvir, naux));
  const bool fock = opts && opts->f_ov;
  const int nin = fock ? 8 : 7;
  const void* ptrs[8] = {eps_occ, eps_vir, t1, t2, B_oo, B_ov, B_vv, fock ? opts->f_ov : nullptr};
  const char* names[8] = {"eps_occ", "eps_vir", "t1", "t2", "B_oo", "B_ov", "B_vv", "opts->f_ov"};
  const size_t o = nocc, v = nvir, X = naux;
  const size_t elems[8] = {o, v, o * v, o * o * v * v, X * o * o, X * o * v, X * v * v, o * v};
  for (int n = 0; n < nin; ++n)
    if (!ptrs[n]) {
      set_error(BQC_ERR_NULL_POINTER, "%s is NULL", names[n]);
      return BQC_ERR_NULL_POINTER;
    }
  if (!e_total_host) {
    set_error(BQC_ERR_NULL_POINTER, "e_total_host is NULL");
    return BQC_ERR_NULL_POINTER;
  }
  size_t total = 0, offs[8];
  for (int n = 0; n < nin; ++n) { offs[n] = total; total += round_up(elems[n] * 8, 256); }
  const bool abc = opts && (opts->flags & BQC_T_FLAG_ABC_DRIVEN);
  const size_t ntrip = num_triplets(abc ? nvir : nocc);
  const size_t off_trip = total;
  total += round_up(ntrip * 8, 256);
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
  // An occupied window [lo,hi) of the ijk-driven schedule reads t2 only through rows t2[x,:,:,:], lo <= x < hi
  // (B~ rows, hole columns, Fock tiles): copy just that contiguous slice; the rest of the device buffer is
  // never read.  The abc-driven schedule transposes all of t2 and takes the whole array.
  size_t t2_first = 0, t2_count = elems[3];
  if (!abc) {
    int lo = 0, hi = nocc;
    if (resolve_window(nocc, opts, &lo, &hi) != BQC_OK) {
      cudaFree(dev);
      return g_err;
    }
    t2_first = (size_t)lo * o * v * v;
    t2_count = (size_t)(hi - lo) * o * v * v;
  }
  for (int n = 0; n < nin && rc == BQC_OK; ++n) {
    const size_t first = n == 3 ? t2_first : 0, count = n == 3 ? t2_count : elems[n];
    cudaError_t e = cudaMemcpyAsync(dev + offs[n] + first * 8, static_cast<const double*>(ptrs[n]) + first,
                                    count * 8, cudaMemcpyHostToDevice, stream);
    if (e != cudaSuccess) {
      set_error(BQC_ERR_CUDA, "H2D copy of %s failed: %s", names[n], cudaGetErrorString(e));
      rc = BQC_ERR_CUDA;
    }
    h2d += count * 8;
  }
  if (rc == BQC_OK) {
    auto D = [&](int n) { return reinterpret_cast<const double*>(dev + offs[n]); };
    bqc_t_opts dopts;
    memset(&dopts, 0, sizeof(dopts));
    if (opts) dopts = *opts;
    dopts.f_ov = fock ? D(7) : nullptr;   // the device copy replaces the caller's host pointer
    rc = bqc_t_energy_ex(nocc, nvir, naux, D(0), D(1), D(2), D(3), D(4), D(5), D(6), &dopts, nullptr, 0,
                         e_total_host, e_triplet_host ? reinterpret_cast<double*>(dev + off_trip) : nullptr,
                         stream);
  }
  size_t d2h = 8;
  if (rc == BQC_OK && e_triplet_host) {
    cudaError_t e = cudaMemcpyAsync(e_triplet_host, dev + off_trip, ntrip * 8, cudaMemcpyDeviceToHost, stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(stream);
    if (e != cudaSuccess) {
      set_error(BQC_ERR_CUDA, "D2H copy of e_triplet failed: %s", cudaGetErrorString(e));
      rc = BQC_ERR_CUDA;
    }
    d2h += ntrip * 8;
  }
  cudaFree(dev);
  if (h2d_bytes) *h2d_bytes = h2d;
  if (d2h_bytes) *d2h_bytes = d2h;
  return rc;
}

int bqc_t_debug_slabs(int nocc, int nvir, int naux, const double* t2, const double* B_oo, const double* B_ov,
                      const double* B_vv, int x, int y, double* I_dev, double* O_dev, double* J_dev,
                      void* stream_v) {
  clear_error();
  cudaStream_t stream = static_cast<cudaStream_t>(stream_v);
  BQC_TRY(check_sizes(nocc, nvir, naux));
  BQC_TRY(check_device());
  if (x < 0 || x >= nocc || y < 0 || y >= nocc) {
    set_error(BQC_ERR_INVALID_SIZE, "x=%d y=%d outside [0,%d)", x, y, nocc);
    return BQC_ERR_INVALID_SIZE;
  }
  BQC_TRY(check_device_ptr(t2, "t2"));
  BQC_TRY(check_device_ptr(B_oo, "B_oo"));
  BQC_TRY(check_device_ptr(B_ov, "B_ov"));
  BQC_TRY(check_device_ptr(B_vv, "B_vv"));
  Inputs in = {nullptr, nullptr, nullptr, t2, B_oo, B_ov, B_vv};
  std::vector<int> act;
  act.push_back(std::min(x, y));
  if (x != y) act.push_back(std::max(x, y));
  bqc_t_opts o2;
  memset(&o2, 0, sizeof(o2));
  o2.max_batch = 1;
  o2.occ_block = 2;
  Pipeline p;
  BQC_TRY(p.setup(nocc, nvir, naux, in, act, &o2, nullptr, 0, stream));
  BQC_TRY(p.build_schedule());
  p.actions.clear();
  BQC_TRY(p.prepare());
  Ctx& c = p.c;
  const Plan& P = c.P;
  const int px = (int)(std::find(act.begin(), act.end(), x) - act.begin());
  const int py = (int)(std::find(act.begin(), act.end(), y) - act.begin());
  const int v = nvir;
  if (I_dev) {
    BQC_TRY(check_device_ptr(I_dev, "I_dev"));
    BQC_TRY(p.form_block(0, 0, stream));   // one block holds all active orbitals (na <= 2 <= Bo)
    BQC_TRY(launch_copy3(c.slabs() + (size_t)px * P.slab_elems, (long long)v * P.Kp, P.Kp, 1, I_dev, v, v, v,
                         stream));
  }
  if (O_dev) {
    BQC_TRY(check_device_ptr(O_dev, "O_dev"));
    // O_xy[l,u] = (x u|y l) = B~_xy[u, v + l]  -> out[l][u]
    BQC_TRY(launch_copy3(c.btil() + ((size_t)px * P.na + py) * v * P.Kp + v, 0, 1, P.Kp, O_dev, 1, nocc, v,
                         stream));
  }
  if (J_dev) {
    BQC_TRY(check_device_ptr(J_dev, "J_dev"));
    BQC_CUDA_OK(cudaMemcpyAsync(J_dev, c.J() + ((size_t)px * P.na + py) * v * v, (size_t)v * v * 8,
                                cudaMemcpyDeviceToDevice, stream));
  }
  BQC_CUDA_OK(cudaStreamSynchronize(stream));
  BQC_CUDA_OK(cudaStreamSynchronize(c.s_form));
  return BQC_OK;
}

int bqc_t_debug_wv(int nocc, int nvir, int naux, const double* eps_occ, const double* eps_vir,
                   const double* t1, const double* t2, const double* B_oo, const double* B_ov,
                   const double* B_vv, const double* f_ov, int i, int j, int k, double* W_dev, double* V_dev,
                   void* stream_v) {
  clear_error();
  cudaStream_t stream = static_cast<cudaStream_t>(stream_v);
  Inputs in = {eps_occ, eps_vir, t1, t2, B_oo, B_ov, B_vv, f_ov};
  BQC_TRY(validate_inputs(nocc, nvir, naux, in));
  if (f_ov) BQC_TRY(check_device_ptr(f_ov, "f_ov"));
  if (i < 0 || j < 0 || k < 0 || i >= nocc || j >= nocc || k >= nocc) {
    set_error(BQC_ERR_INVALID_SIZE, "triplet (%d,%d,%d) outside [0,%d)", i, j, k, nocc);
    return BQC_ERR_INVALID_SIZE;
  }
  if (W_dev) BQC_TRY(check_device_ptr(W_dev, "W_dev"));
  if (V_dev) BQC_TRY(check_device_ptr(V_dev, "V_dev"));
  std::vector<int> act = {i, j, k};
  std::sort(act.begin(), act.end());
  act.erase(std::unique(act.begin(), act.end()), act.end());
  bqc_t_opts o2;
  memset(&o2, 0, sizeof(o2));
  o2.max_batch = 1;
  o2.occ_block = 3;
  Pipeline p;
  BQC_TRY(p.setup(nocc, nvir, naux, in, act, &o2, nullptr, 0, stream));
  Ctx& c = p.c;
  const Plan& P = c.P;
  // schedule: DF task slots as usual, then the three F tasks of (i,j,k) in the caller's order
  BQC_TRY(p.build_schedule());
  p.actions.clear();
  auto pos = [&](int x) { return (int)(std::find(act.begin(), act.end(), x) - act.begin()); };
  const int pi = pos(i), pj = pos(j), pk = pos(k);
  const size_t task0 = c.tasks.size();
  {
    auto pair = [&](int pz, int py) { return pz * P.na + py; };
    auto f_task = [&](int px, int py, int pz, int cls) {
      GemmTask g;
      memset(&g, 0, sizeof(g));
      g.nterms = 2;
      g.term[0].a_idx = px; g.term[0].a_transposed = 0; g.term[0].b_idx = pair(pz, py);
      g.term[1].a_idx = py; g.term[1].a_transposed = 1; g.term[1].b_idx = pair(pz, px);
      g.c_off = (long long)(cls * P.fsz);
      c.tasks.push_back(g);
    };
    f_task(pi, pj, pk, 0);
    f_task(pi, pk, pj, 1);
    f_task(pj, pk, pi, 2);
  }
  BQC_TRY(p.prepare());
  BQC_TRY(p.form_block(0, 0, stream));
  GemmParams prm;
  memset(&prm, 0, sizeof(prm));
  prm.ntasks = 3;
  prm.tasks = c.tasks_dev() + task0;
  prm.C = c.F();
  BQC_TRY(launch_f_gemm(c, prm, stream));
  BQC_TRY(launch_assemble_wv(c.F(), P.nbv, nvir, c.J(), P.na, pi, pj, pk, t1 + (size_t)i * nvir,
                             t1 + (size_t)j * nvir, t1 + (size_t)k * nvir, t2, nocc, i, j, k, f_ov, W_dev, V_dev,
                             stream));
  BQC_CUDA_OK(cudaStreamSynchronize(stream));
  BQC_CUDA_OK(cudaStreamSynchronize(c.s_form));
  return BQC_OK;
}

int bqc_debug_tiling(int nvir, int* out, int n) {
  clear_error();
  if (nvir <= 0 || !out || n < 14) {
    set_error(BQC_ERR_INVALID_SIZE, "bqc_debug_tiling: nvir=%d, out=%p, n=%d (need 14)", nvir, (void*)out, n);
    return -1;
  }
  NSegment ns[2];
  MSegment ms[2];
  const int nn = split_n(nvir, ns), nm = split_m(nvir, nvir, ms);
  for (int k = 0; k < 14; ++k) out[k] = 0;
  for (int k = 0; k < nn; ++k) { out[3 * k] = ns[k].n0; out[3 * k + 1] = ns[k].ntiles; out[3 * k + 2] = ns[k].nf; }
  for (int k = 0; k < nm; ++k) {
    out[6 + 4 * k] = ms[k].m1_0; out[7 + 4 * k] = ms[k].tiles_m1; out[8 + 4 * k] = ms[k].tp;
    out[9 + 4 * k] = 1 << ms[k].tq_log2;
  }
  return nn * 10 + nm;
}

int bqc_dgemm_nt(int M, int N, int K, const double* A, int lda, const double* B, int ldb, double* C, int ldc,
                 void* stream_v) {
  clear_error();
  cudaStream_t stream = static_cast<cudaStream_t>(stream_v);
  if (M <= 0 || N <= 0 || K <= 0 || lda < K || ldb < K || ldc < N || (lda & 1) || (ldb & 1)) {
    set_error(BQC_ERR_INVALID_SIZE, "bqc_dgemm_nt: M=%d N=%d K=%d lda=%d ldb=%d ldc=%d", M, N, K, lda, ldb, ldc);
    return BQC_ERR_INVALID_SIZE;
  }
  BQC_TRY(check_device());
  BQC_TRY(check_device_ptr(A, "A"));
  BQC_TRY(check_device_ptr(B, "B"));
  BQC_TRY(check_device_ptr(C, "C"));
  if ((reinterpret_cast<uintptr_t>(A) & 15) || (reinterpret_cast<uintptr_t>(B) & 15)) {
    set_error(BQC_ERR_MISALIGNED, "bqc_dgemm_nt: A and B must be 16-byte aligned");
    return BQC_ERR_MISALIGNED;
  }
  const int nf = choose_nf(N);
  CUtensorMap tA, tB;
  {
    const unsigned long long dA[4] = {(unsigned long long)K, (unsigned long long)M, 1, 1};
    const unsigned long long sA[4] = {8, (unsigned long long)lda * 8, (unsigned long long)lda * 8 * M,
                                      (unsigned long long)lda * 8 * M};
    BQC_TRY(make_tensor_map_f64(&tA, A, dA, sA, 128, 1));
    const unsigned long long dB[4] = {(unsigned long long)K, (unsigned long long)N, 1, 1};
    const unsigned long long sB[4] = {8, (unsigned long long)ldb * 8, (unsigned long long)ldb * 8 * N,
                                      (unsigned long long)ldb * 8 * N};
    BQC_TRY(make_tensor_map_f64(&tB, B, dB, sB, gemm_bn(nf), 1));
  }
  GemmTask task = single_term_task(0);
  GemmTask* task_dev = nullptr;
  BQC_CUDA_OK(cudaMalloc(&task_dev, sizeof(GemmTask)));
  cudaError_t e = cudaMemcpyAsync(task_dev, &task, sizeof(task), cudaMemcpyHostToDevice, stream);
  int rc = BQC_OK;
  if (e != cudaSuccess) {
    set_error(BQC_ERR_CUDA, "task upload failed: %s", cudaGetErrorString(e));
    rc = BQC_ERR_CUDA;
  }
  if (rc == BQC_OK) {
    GemmParams prm;
    memset(&prm, 0, sizeof(prm));
    prm.ntasks = 1;
    prm.tp = 1; prm.tq_log2 = 7;
    prm.tiles_m1 = 1;
    prm.tiles_m2 = ceil_div(M, 128);
    prm.tiles_n = ceil_div(N, gemm_bn(nf));
    prm.m1_ext = 1; prm.m2_ext = M; prm.n_ext = N;
    prm.kiters = ceil_div(K, kBK);
    prm.out_mode = 0;
    prm.n2_ext = INT_MAX;
    prm.sM1 = 0; prm.sM2 = ldc; prm.sN1 = 0; prm.sN2 = 1;
    prm.tasks = task_dev;
    prm.C = C;
    rc = launch_gemm_nt(nf, tA, tA, tB, prm, stream);
  }
  if (rc == BQC_OK) {
    e = cudaStreamSynchronize(stream);
    if (e != cudaSuccess) {
      set_error(BQC_ERR_CUDA, "bqc_dgemm_nt kernel failed: %s", cudaGetErrorString(e));
      rc = BQC_ERR_CUDA;
    }
  }
  cudaFree(task_dev);
  return rc;
}

double bqc_fp64_peak_tflops(int kind, double seconds, void* stream) {
  clear_error();
  if (kind < 0 || kind > 2 || !(seconds > 0.0)) {
    set_error(BQC_ERR_INVALID_OPTION, "bqc_fp64_peak_tflops: kind=%d seconds=%g", kind, seconds);
    return -1.0;
  }
  if (check_device() != BQC_OK) return -1.0;
  return run_fp64_peak(kind, seconds, static_cast<cudaStream_t>(stream));
}

}  // extern "C"
