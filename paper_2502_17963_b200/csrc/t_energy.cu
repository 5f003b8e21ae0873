// t_energy.cu — the triplet-block scheduler ("engine") and the C ABI of the (T) energy.
//
// How W is built:
//   augmented slab   I~_x[p,q,kappa] : kappa <  v      -> (x p|q d)                 (DF slab former, a1)
//                                      kappa = v + l   -> -t2[x,l,p,q]              (hole columns)
//   augmented pair   B~_zy[r,kappa]  : kappa <  v      -> t2[z,y,r,d]
//                                      kappa = v + l   -> (z r|y l)                 (DF slab former, a1)
//   F(x,y,z)[p,q,r] = sum_kappa I~_x[p,q,kappa] B~_zy[r,kappa] + sum_kappa I~_y[q,p,kappa] B~_zx[r,kappa]
//   W_ijk[a,b,c]    = F(i,j,k)[a,b,c] + F(i,k,j)[a,c,b] + F(j,k,i)[b,c,a]          (= PAPER.md Eq. (2), G1/G5)
// i.e. the six particle and six hole contractions of Eq. (2) become six K = v+o tile-GEMM terms.
//
// What is resident: the outer orbitals are cut into blocks of Bo; block triples I <= J <= K are
// walked in order with a cache of 4 slab sets (I -> set 0, J -> set 1, K alternating 2/3) formed on a second
// stream, and the B~ / J pair blocks of the set pairs a block triple touches, formed on the main stream just
// before their first use.  Nothing scales with (outer extent)^2: the full (vv|ov), (ov|ov) and B~ tensors are
// never stored.  The abc-driven schedule is the same engine on the particle-hole dual problem
// (Plan::dual), reading the caller's arrays through dual-aware packing kernels — no transposed copy of t2.
#include <limits.h>
#include <math.h>
#include <stdarg.h>
#include <string.h>

#include <algorithm>
#include <memory>
#include <vector>

#include "gemm_nt.cuh"
#include "kernels.cuh"
#include "plan.cuh"

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

// caller-space device pointers (never dualised: the packing kernels read them as they are)
struct Inputs {
  const double *eps_occ, *eps_vir, *t1, *t2, *B_oo, *B_ov, *B_vv;
  const double* f_ov = nullptr;   // optional occupied-virtual Fock block (bqc_t_opts.f_ov)
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
  long long sM1, sM2, sN1, sN2; int n2_ext;
  double* C;                                // output base (element (0,0,0) of this GEMM)
};

struct Action {
  enum Kind { FORM, PAIR, TRIPLE } kind;
  int set, block;                 // FORM: slab set <- block.  PAIR: first set / block (z).  TRIPLE: unused
  int set2, block2;               // PAIR: second set / block (y)
  int need_j, need_panel;         // PAIR: also form J; (re)build the K-major panel of block2
  int I, J, K, sJ, sK;            // TRIPLE: the block triple and the slab sets of its J and K blocks (I: set 0)
};

// ------------------------------------------------------------------ the engine
// Everything that does not depend on the values of the inputs: plan, workspace, helper stream, events,
// tensor maps and the host-built schedule.  Reused across calls with the same sizes/options (see engine_for).
struct Engine {
  Plan P;
  int nocc = 0, nvir = 0, naux = 0;   // caller space
  bqc_t_opts key_opts;                // options the engine was built for (f_ov reduced to NULL / non-NULL)
  void* key_ws = nullptr;             // caller workspace the engine was built on (NULL: owns its own)
  size_t key_ws_bytes = 0;
  int device = -1;
  Inputs in;
  uint8_t* ws = nullptr;
  bool own_ws = false;
  cudaStream_t s_main = nullptr, s_form = nullptr, s_cap = nullptr;
  cudaEvent_t ev_formed[4] = {}, ev_free[4] = {}, ev_fork = nullptr, ev_join = nullptr;
  bool ev_free_valid[4] = {};
  // F-GEMM configuration
  MSegment f_mseg[2];                // row segments of the F GEMM (split_m): main tiles + remainder strip
  int f_nmseg = 0;
  NSegment f_seg[2];                 // column segments of the F GEMM (split_n): exact cover of v up to 16
  int f_nseg = 0;
  CUtensorMap tm_slab[2], tm_slabT[2], tm_btil[2];
  // host schedule: the action list (slab-set / pair-block formations and block triples, in order); the
  // triplet records and F-GEMM tasks of a block triple are generated when it is reached, into one of two
  // pinned chunks, and uploaded into the matching device chunk (so nothing of size #triplets lives anywhere)
  std::vector<int> orbits;
  std::vector<Action> actions;
  std::vector<int> bt_owner;         // BQC_T_FLAG_SHARD_BLOCKS: owner of every block triple
  size_t ncompute = 0;               // W-builder launches of the whole schedule
  GemmTask df_task;                  // the one task of every DF GEMM (single term, c_off 0)
  uint8_t* pinned = nullptr;         // 2 chunks: [chunk_trips TripletRec][3 chunk_trips GemmTask], then the
                                     // orbit table and the DF task (static tables uploaded every call)
  // CUDA graph of a short schedule (launch-bound regime): the whole call — repacking, slab and
  // pair formation, W builder, energy kernels, sums — captured once per set of argument pointers and replayed
  cudaGraphExec_t graph_exec = nullptr;
  const void* graph_key[10] = {};
  long long graph_launches = 0;
  size_t ntriple_actions = 0;
  bool capturing = false;
  cudaEvent_t ev_up[2] = {};         // upload of chunk b has executed: its pinned half may be rewritten
  bool ev_up_valid[2] = {};
  int chunk_next = 0;
  // BQC_T_FLAG_PROFILE: timing events (pooled, reused across calls)
  std::vector<cudaEvent_t> ev_pool;
  size_t ev_used = 0;
  std::vector<cudaEvent_t> prof_main;   // [3n] before W builder, [3n+1] after it, [3n+2] after the energy kernels
  std::vector<cudaEvent_t> prof_form;   // [2n], [2n+1] around each slab-block / pair-block formation
  cudaEvent_t prof_begin = nullptr, prof_prepared = nullptr, prof_end = nullptr;

  int prof_mark(std::vector<cudaEvent_t>& v, cudaStream_t s) {
    if (ev_used == ev_pool.size()) {
      cudaEvent_t e;
      BQC_CUDA_OK(cudaEventCreate(&e));
      ev_pool.push_back(e);
    }
    cudaEvent_t e = ev_pool[ev_used++];
    v.push_back(e);
    BQC_CUDA_OK(cudaEventRecord(e, s));
    return BQC_OK;
  }

  double* d(size_t off) const { return reinterpret_cast<double*>(ws + off); }
  double* btvv() const { return d(P.off_btvv); }
  double* btov() const { return d(P.off_btov); }
  double* panel() const { return d(P.off_panel); }
  double* btil() const { return d(P.off_btil); }
  double* J() const { return d(P.off_J); }
  double* slabs() const { return d(P.off_slabs); }
  double* F() const { return d(P.off_F); }
  double* partial() const { return d(P.off_partial); }
  double* etrip() const { return d(P.off_etrip); }
  double* esum() const { return d(P.off_esum); }
  int* orbits_dev() const { return reinterpret_cast<int*>(ws + P.off_orbits); }
  GemmTask* df_task_dev() const { return reinterpret_cast<GemmTask*>(ws + P.off_tasks); }
  // device chunk b: F tasks follow the DF task slot(s) at off_tasks
  GemmTask* tasks_dev(int b) const { return df_task_dev() + 8 + (size_t)b * 3 * P.chunk_trips; }
  TripletRec* trips_dev(int b) const { return reinterpret_cast<TripletRec*>(ws + P.off_trips) + (size_t)b * P.chunk_trips; }
  size_t pinned_chunk_bytes() const { return P.chunk_trips * (sizeof(TripletRec) + 3 * sizeof(GemmTask)); }
  int* orbits_host() const { return reinterpret_cast<int*>(pinned + 2 * pinned_chunk_bytes()); }
  GemmTask* df_task_host() const { return reinterpret_cast<GemmTask*>(pinned + 2 * pinned_chunk_bytes() + round_up((size_t)P.norbits * 4, 64)); }
  bool graph_eligible() const { return !P.profile && ncompute <= 8 && ntriple_actions <= 2 && actions.size() <= 24; }
  int enqueue(double* e_triplet_dev, cudaStream_t stream);
  TripletRec* trips_host(int b) const { return reinterpret_cast<TripletRec*>(pinned + (size_t)b * pinned_chunk_bytes()); }
  GemmTask* tasks_host(int b) const { return reinterpret_cast<GemmTask*>(trips_host(b) + P.chunk_trips); }
  // pipeline-space views of the small inputs (dual copies live in the workspace)
  const double* eps_o() const { return P.dual ? d(P.off_small + P.small_eo) : in.eps_occ; }
  const double* eps_v() const { return P.dual ? d(P.off_small + P.small_ev) : in.eps_vir; }
  const double* t1p() const { return P.dual ? d(P.off_small + P.small_t1) : in.t1; }
  const double* fp() const { return !in.f_ov ? nullptr : (P.dual ? d(P.off_small + P.small_f) : in.f_ov); }
  // pipeline-space DF blocks: inner-inner, outer-outer (the caller's arrays, Q-major)
  const double* B_inner() const { return P.dual ? in.B_oo : in.B_vv; }
  const double* B_outer() const { return P.dual ? in.B_vv : in.B_oo; }

  int block_begin(int b) const { return b * P.Bo; }
  int block_end(int b) const { return std::min(P.na, (b + 1) * P.Bo); }
  int slot_of(int pos, int set, int block) const { return set * P.Bo + (pos - block_begin(block)); }

  int init(int nocc_, int nvir_, int naux_, const bqc_t_opts* opts, void* workspace, size_t workspace_bytes,
           const std::vector<int>* act_override);
  int build_schedule();
  int run_df_gemm(const DfGemm& g, cudaStream_t s);
  int launch_f_gemm(GemmParams prm, cudaStream_t s);
  int prepare(cudaStream_t s);
  int exec_form(int set, int block, cudaStream_t s);
  int exec_pair(const Action& a, cudaStream_t s);
  size_t list_triple(const Action& a, TripletRec* trips, GemmTask* tasks) const;
  int exec_triple(const Action& a, cudaStream_t s);
  int exec_compute(int chunk, size_t trip0, size_t ntrip, cudaStream_t s);
  int execute();
  int run(const Inputs& inputs, double* e_total_host, double* e_triplet_dev, cudaStream_t stream);

  ~Engine() {
    for (cudaEvent_t e : ev_pool) cudaEventDestroy(e);
    if (prof_begin) cudaEventDestroy(prof_begin);
    if (prof_prepared) cudaEventDestroy(prof_prepared);
    if (prof_end) cudaEventDestroy(prof_end);
    for (int s = 0; s < 4; ++s) {
      if (ev_formed[s]) cudaEventDestroy(ev_formed[s]);
      if (ev_free[s]) cudaEventDestroy(ev_free[s]);
    }
    if (ev_fork) cudaEventDestroy(ev_fork);
    if (ev_join) cudaEventDestroy(ev_join);
    for (int b = 0; b < 2; ++b)
      if (ev_up[b]) cudaEventDestroy(ev_up[b]);
    if (s_form) cudaStreamDestroy(s_form);
    if (graph_exec) cudaGraphExecDestroy(graph_exec);
    if (pinned) cudaFreeHost(pinned);
    if (own_ws && ws) cudaFree(ws);
  }
};

int Engine::init(int nocc_, int nvir_, int naux_, const bqc_t_opts* opts, void* workspace,
                 size_t workspace_bytes, const std::vector<int>* act_override) {
  nocc = nocc_; nvir = nvir_; naux = naux_;
  memset(&key_opts, 0, sizeof(key_opts));
  if (opts) key_opts = *opts;
  key_ws = workspace;
  key_ws_bytes = workspace_bytes;
  BQC_CUDA_OK(cudaGetDevice(&device));
  if (act_override)
    BQC_TRY(make_plan(P, nocc, nvir, naux, false, *act_override, opts));
  else
    BQC_TRY(make_plan_for(P, nocc, nvir, naux, opts));
  if (workspace) {
    if (workspace_bytes < P.total || (reinterpret_cast<uintptr_t>(workspace) & 255)) {
      set_error(BQC_ERR_WORKSPACE, "workspace of %zu bytes (need %zu, 256-byte aligned; largest buffer: %s, %zu bytes)",
                workspace_bytes, P.total, P.biggest_name, P.biggest_bytes);
      return BQC_ERR_WORKSPACE;
    }
    ws = static_cast<uint8_t*>(workspace);
  } else {
    void* p = nullptr;
    cudaError_t e = cudaMalloc(&p, P.total);
    if (e != cudaSuccess) {
      cudaGetLastError();
      size_t fr = 0, tot = 0;
      cudaMemGetInfo(&fr, &tot);
      set_error(BQC_ERR_WORKSPACE,
                "cudaMalloc of %zu workspace bytes failed (%s; %zu bytes free); largest buffer: %s, %zu bytes — "
                "lower opts.workspace_gib or opts.occ_block / max_batch",
                P.total, cudaGetErrorString(e), fr, P.biggest_name, P.biggest_bytes);
      return BQC_ERR_WORKSPACE;
    }
    ws = static_cast<uint8_t*>(p);
    own_ws = true;
  }
  BQC_CUDA_OK(cudaStreamCreateWithFlags(&s_form, cudaStreamNonBlocking));
  for (int s = 0; s < 4; ++s) {
    BQC_CUDA_OK(cudaEventCreateWithFlags(&ev_formed[s], cudaEventDisableTiming));
    BQC_CUDA_OK(cudaEventCreateWithFlags(&ev_free[s], cudaEventDisableTiming));
  }
  BQC_CUDA_OK(cudaEventCreateWithFlags(&ev_fork, cudaEventDisableTiming));
  BQC_CUDA_OK(cudaEventCreateWithFlags(&ev_join, cudaEventDisableTiming));
  for (int b = 0; b < 2; ++b) BQC_CUDA_OK(cudaEventCreateWithFlags(&ev_up[b], cudaEventDisableTiming));
  BQC_CUDA_OK(cudaMallocHost(&pinned, 2 * pinned_chunk_bytes() + round_up((size_t)P.norbits * 4, 64) + sizeof(GemmTask)));
  df_task = single_term_task(0);

  const int v = P.v;
  f_nmseg = split_m(v, v, f_mseg);
  f_nseg = split_n(v, f_seg);
  for (int m = 0; m < f_nmseg; ++m) {
    const int tq = 1 << f_mseg[m].tq_log2;
    BQC_TRY(tmap(&tm_slab[m], slabs(), P.Kp, v, v, P.nslots, tq, f_mseg[m].tp));
    BQC_TRY(tmap(&tm_slabT[m], slabs(), P.Kp, v, v, P.nslots, 1, tq));
  }
  for (int n = 0; n < f_nseg; ++n)
    BQC_TRY(tmap(&tm_btil[n], btil(), P.Kp, v, (unsigned long long)P.nslots * P.nslots, 1, gemm_bn(f_seg[n].nf), 1));
  // orbit table A <= B <= C of 8-blocks of the inner index
  orbits.reserve(P.norbits);
  for (int A = 0; A < P.nbv; ++A)
    for (int B = A; B < P.nbv; ++B)
      for (int C = B; C < P.nbv; ++C) orbits.push_back(A | (B << 10) | (C << 20));
  memcpy(orbits_host(), orbits.data(), orbits.size() * 4);
  *df_task_host() = df_task;
  return build_schedule();
}

// Triplet records (and, if tasks != NULL, the three F-GEMM tasks of each) of block triple `a` owned by this
// shard, in loop order.  Returns their number.
size_t Engine::list_triple(const Action& a, TripletRec* trips, GemmTask* tasks) const {
  size_t n = 0;
  for (int pi = block_begin(a.I); pi < block_end(a.I); ++pi)
    for (int pj = std::max(pi, block_begin(a.J)); pj < block_end(a.J); ++pj)
      for (int pk = std::max(pj, block_begin(a.K)); pk < block_end(a.K); ++pk) {
        if (pi == pj && pj == pk) continue;   // g(i,i,i) = 0 exactly
        TripletRec t;
        t.i = P.act[pi]; t.j = P.act[pj]; t.k = P.act[pk];
        t.pi = slot_of(pi, 0, a.I); t.pj = slot_of(pj, a.sJ, a.J); t.pk = slot_of(pk, a.sK, a.K);
        t.index = (long long)triplet_index(P.o, t.i, t.j, t.k);
        if (!P.shard_blocks && (int)(t.index % P.shard_count) != P.shard_rank) continue;
        if (trips) trips[n] = t;
        if (tasks) {
          const size_t in_batch = n % (size_t)P.nbatch;   // F arrays are indexed within a W-builder launch
          auto pair = [&](int sz, int sy) { return sz * P.nslots + sy; };
          // F(x,y,z): term0 = (I~_x, canonical rows, B~_zy), term1 = (I~_y, transposed rows, B~_zx)
          auto f_task = [&](int sx, int sy, int sz, int cls) {
            GemmTask& g = tasks[3 * n + cls];
            memset(&g, 0, sizeof(g));
            g.nterms = 2;
            g.term[0].a_idx = sx; g.term[0].a_transposed = 0; g.term[0].b_idx = pair(sz, sy);
            g.term[1].a_idx = sy; g.term[1].a_transposed = 1; g.term[1].b_idx = pair(sz, sx);
            g.c_off = (long long)((in_batch * 3 + cls) * P.fsz);
          };
          f_task(t.pi, t.pj, t.pk, 0);   // F(i,j,k)
          f_task(t.pi, t.pk, t.pj, 1);   // F(i,k,j)
          f_task(t.pj, t.pk, t.pi, 2);   // F(j,k,i)
        }
        ++n;
      }
  return n;
}

int Engine::build_schedule() {
  const int Bo = P.Bo;
  actions.clear();
  ncompute = 0;
  ntriple_actions = 0;

  // ---- block triples I <= J <= K with the slot-set protocol: I -> set 0, J -> set 1, K -> sets 2/3
  int set_block[4] = {-1, -1, -1, -1};
  struct PairTag { int bz = -1, by = -1, has_j = 0; } tag[4][4];
  int panel_block = -1;
  int kflip = 0;
  auto acquire = [&](int set, int block) {
    if (set_block[set] == block) return;
    Action a;
    memset(&a, 0, sizeof(a));
    a.kind = Action::FORM; a.set = set; a.block = block;
    actions.push_back(a);
    set_block[set] = block;
  };
  const bool single_run_blocks = (P.nruns == 1);

  long long block_triple = -1;
  bt_owner.clear();
  if (P.shard_blocks) bt_owner = deal_block_triples(P.na, Bo, P.shard_count);
  for (int I = 0; I < P.nblk; ++I) {
    for (int Jb = I; Jb < P.nblk; ++Jb) {
      const int sJ = (Jb == I) ? 0 : 1;
      for (int K = Jb; K < P.nblk; ++K) {
        ++block_triple;
        // BQC_T_FLAG_SHARD_BLOCKS: whole block triples are dealt to the shards, so a shard forms only the
        // slabs of its own block triples; otherwise every shard owns some triplets of every block triple
        if (P.shard_blocks && bt_owner[(size_t)block_triple] != P.shard_rank) continue;
        int sK = sJ;
        if (K != Jb) sK = (set_block[2] == K) ? 2 : (set_block[3] == K ? 3 : 2 + (kflip & 1));
        Action t;
        memset(&t, 0, sizeof(t));
        t.kind = Action::TRIPLE;
        t.I = I; t.J = Jb; t.K = K; t.sJ = sJ; t.sK = sK;
        // triplets of this block triple owned by this shard (every one, unless the per-triplet modulo shards)
        const size_t ntr = (P.shard_count > 1 && !P.shard_blocks) ? list_triple(t, nullptr, nullptr)
                                                                  : (size_t)block_triple_work(P.na, Bo, I, Jb, K);
        if (ntr == 0) continue;
        if (ntr > P.chunk_trips) {
          set_error(BQC_ERR_WORKSPACE, "internal: block triple of %zu triplets exceeds the chunk of %zu", ntr,
                    P.chunk_trips);
          return BQC_ERR_WORKSPACE;
        }
        if (K != Jb && sK >= 2 && set_block[sK] != K) ++kflip;
        // slabs are formed only for block triples that have work (the acquire calls are idempotent)
        acquire(0, I);
        if (Jb != I) acquire(1, Jb);
        if (K != Jb) acquire(sK, K);
        // B~ / J pair blocks of the ordered set pairs this block triple touches
        const int sets[3] = {0, sJ, sK}, blks[3] = {I, Jb, K};
        for (int p = 0; p < 3; ++p)
          for (int q = 0; q < 3; ++q) {
            if (p == q) continue;
            const int sz = sets[p], sy = sets[q];
            const int want_j = (p < q) ? 1 : 0;   // J_ij, J_ik, J_jk: the earlier orbital first
            PairTag& tg = tag[sz][sy];
            if (tg.bz == blks[p] && tg.by == blks[q] && (tg.has_j || !want_j)) continue;
            // when the same set pair comes again in this loop as an (earlier, later) pair it wants J: form it now
            int need_j = want_j;
            for (int p2 = 0; p2 < 3; ++p2)
              for (int q2 = p2 + 1; q2 < 3; ++q2)
                if (sets[p2] == sz && sets[q2] == sy) need_j = 1;
            Action a;
            memset(&a, 0, sizeof(a));
            a.kind = Action::PAIR;
            a.set = sz; a.block = blks[p]; a.set2 = sy; a.block2 = blks[q];
            a.need_j = need_j;
            a.need_panel = !(single_run_blocks && panel_block == blks[q]);
            panel_block = single_run_blocks ? blks[q] : -1;
            actions.push_back(a);
            tg.bz = blks[p]; tg.by = blks[q]; tg.has_j = need_j;
          }
        actions.push_back(t);
        ++ntriple_actions;
        ncompute += (ntr + P.nbatch - 1) / P.nbatch;
      }
    }
  }
  return BQC_OK;
}

int Engine::run_df_gemm(const DfGemm& g, cudaStream_t s) {
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
  prm.ktail8 = (P.X - (prm.kiters - 1) * kBK) <= 8;
  prm.out_mode = 0;
  prm.n2_ext = g.n2_ext;
  prm.sM1 = g.sM1; prm.sM2 = g.sM2; prm.sN1 = g.sN1; prm.sN2 = g.sN2;
  prm.tasks = df_task_dev();   // single term, a_idx = b_idx = 0, c_off = 0
  prm.C = g.C;
  return launch_gemm_nt(nf, tA, tA, tB, prm, s);
}

// The W-builder GEMM of `prm.ntasks` tasks: one launch per (row segment, column segment).
int Engine::launch_f_gemm(GemmParams prm, cudaStream_t s) {
  const int v = P.v;
  prm.m1_ext = v; prm.m2_ext = v; prm.n_ext = v;
  prm.kiters = P.Kp / kBK;
  prm.ktail8 = (P.v + P.o - (prm.kiters - 1) * kBK) <= 8;   // columns [v+o, Kp) are zero
  prm.out_mode = 1;
  prm.nbv = P.nbv;
  prm.n2_ext = 1;
  for (int m = 0; m < f_nmseg; ++m) {
    const MSegment& ms = f_mseg[m];
    prm.tp = ms.tp; prm.tq_log2 = ms.tq_log2;
    prm.tiles_m1 = ms.tiles_m1;
    prm.tiles_m2 = ceil_div(v, 1 << ms.tq_log2);
    prm.m1_base = prm.m1_out = ms.m1_0;
    for (int n = 0; n < f_nseg; ++n) {
      prm.tiles_n = f_seg[n].ntiles;
      prm.n_base = prm.n_out = f_seg[n].n0;
      BQC_TRY(launch_gemm_nt(f_seg[n].nf, tm_slab[m], tm_slabT[m], tm_btil[n], prm, s));
    }
  }
  return BQC_OK;
}

// Per-call set-up on the main stream: dual views of the small inputs, K-major copies of the DF factors the
// slab former reads, zero K-padding, the static tables.  Nothing here synchronises the host: the host
// vectors that are uploaded live in the engine.
int Engine::prepare(cudaStream_t s) {
  const int o = P.o, v = P.v, X = P.X;
  if (P.dual) {
    // eps_occ' = -eps_vir, eps_vir' = -eps_occ, t1'[a,i] = t1[i,a], f'[a,i] = -f[i,a]
    BQC_TRY(launch_transpose_scale(in.eps_vir, d(P.off_small + P.small_eo), 1, 1, o, -1.0, s));
    BQC_TRY(launch_transpose_scale(in.eps_occ, d(P.off_small + P.small_ev), 1, 1, v, -1.0, s));
    BQC_TRY(launch_transpose_scale(in.t1, d(P.off_small + P.small_t1), 1, v, o, 1.0, s));
    if (in.f_ov) BQC_TRY(launch_transpose_scale(in.f_ov, d(P.off_small + P.small_f), 1, v, o, -1.0, s));
  }
  // K-major copies: Bt_vv[(q,d)][Q] (inner-inner block), Bt_ov[(x,p)][Q] (outer x, inner p)
  BQC_TRY(launch_transpose_pad(B_inner(), (long long)v * v, 0, (long long)v * v, btvv(), X, P.Xp, 0, 0, s));
  if (!P.dual)
    BQC_TRY(launch_transpose_pad(in.B_ov, (long long)o * v, 0, (long long)o * v, btov(), X, P.Xp, 0, 0, s));
  else   // the caller's B_ov[Q][i][a] has the inner index first: pair-transposed rows
    BQC_TRY(launch_transpose_pad(in.B_ov, (long long)o * v, 0, (long long)o * v, btov(), X, P.Xp, o, v, s));
  // zero fills: the K padding columns [v+o, Kp) of B~ and of the slabs (nobody else writes them), e_ijk
  if (P.Kp > v + o) {
    const size_t w = (size_t)(P.Kp - v - o) * 8, pitch = (size_t)P.Kp * 8;
    BQC_CUDA_OK(cudaMemset2DAsync(btil() + (v + o), pitch, 0, w, (size_t)P.nslots * P.nslots * v, s));
    BQC_CUDA_OK(cudaMemset2DAsync(slabs() + (v + o), pitch, 0, w, (size_t)P.nslots * v * v, s));
  }
  BQC_CUDA_OK(cudaMemsetAsync(etrip(), 0, num_triplets(o) * 8, s));
  // the static tables: orbit table and the DF task (host copies live in the engine; the schedule chunks follow
  // block triple by block triple, see exec_triple)
  BQC_CUDA_OK(cudaMemcpyAsync(orbits_dev(), orbits_host(), orbits.size() * 4, cudaMemcpyHostToDevice, s));
  BQC_CUDA_OK(cudaMemcpyAsync(df_task_dev(), df_task_host(), sizeof(GemmTask), cudaMemcpyHostToDevice, s));
  // the former stream starts after the repacked inputs exist
  BQC_CUDA_OK(cudaEventRecord(ev_fork, s));
  BQC_CUDA_OK(cudaStreamWaitEvent(s_form, ev_fork, 0));
  for (int n = 0; n < 4; ++n) ev_free_valid[n] = false;
  return BQC_OK;
}

// Augmented slabs of one outer block into slot set `set` (row a1 + hole columns).
int Engine::exec_form(int set, int block, cudaStream_t s) {
  const int v = P.v;
  const int p0 = block_begin(block), p1 = block_end(block);
  for (const Run& r : runs_of(P.act, p0, p1)) {
    const int slot0 = slot_of(r.pos0, set, block);
    DfGemm g;
    g.A = btvv(); g.a_d1 = v; g.a_d2 = v;               // rows (m1 = q, m2 = d)
    g.B = btov(); g.b_rows = (long long)P.o * v;        // rows n = (x, p)
    g.m1_base = 0; g.m1_ext = v; g.m2_ext = v;
    g.n_base = r.orb0 * v; g.n_ext = (long long)r.len * v;
    g.sM1 = P.Kp; g.sM2 = 1; g.sN1 = 0; g.sN2 = (long long)v * P.Kp; g.n2_ext = INT_MAX;
    g.C = slabs() + (size_t)slot0 * P.slab_elems;
    BQC_TRY(run_df_gemm(g, s));
    BQC_TRY(launch_slab_holes(in.t2, slabs(), P.o, v, P.Kp, r.orb0, r.len, slot0, P.dual, s));
  }
  return BQC_OK;
}

// B~ (both halves) and, if asked, J of the pair block (set, block) x (set2, block2)   (row a1).
int Engine::exec_pair(const Action& a, cudaStream_t s) {
  const int o = P.o, v = P.v, ns = P.nslots;
  for (const Run& ry : runs_of(P.act, block_begin(a.block2), block_end(a.block2))) {
    // K-major panel of the outer-outer DF block: rows ((y - y0) o + l)[Q] = B_outer[Q][y][l]
    if (a.need_panel || P.nruns > 1)
      BQC_TRY(launch_transpose_pad(B_outer(), (long long)o * o, (long long)ry.orb0 * o, (long long)ry.len * o,
                                   panel(), P.X, P.Xp, 0, 0, s));
    const int sy0 = slot_of(ry.pos0, a.set2, a.block2);
    for (const Run& rz : runs_of(P.act, block_begin(a.block), block_end(a.block))) {
      const int sz0 = slot_of(rz.pos0, a.set, a.block);
      const size_t pair0 = (size_t)sz0 * ns + sy0;
      BQC_TRY(launch_btilde_t2(in.t2, btil(), o, v, P.Kp, ns, rz.orb0, rz.len, ry.orb0, ry.len, sz0, sy0, P.dual, s));
      DfGemm g;   // hole columns: B~_zy[r, v + l] = (z r|y l)
      g.A = btov(); g.a_d1 = v; g.a_d2 = o;
      g.B = panel(); g.b_rows = (long long)ry.len * o;
      g.m1_base = rz.orb0; g.m1_ext = rz.len; g.m2_ext = v;
      g.n_base = 0; g.n_ext = (long long)ry.len * o;
      g.sM1 = (long long)ns * v * P.Kp; g.sM2 = P.Kp; g.sN1 = (long long)v * P.Kp; g.sN2 = 1; g.n2_ext = o;
      g.C = btil() + pair0 * v * P.Kp + v;
      BQC_TRY(run_df_gemm(g, s));
      if (a.need_j) {
        DfGemm j;   // J_zy[u, w] = (z u|y w)
        j.A = btov(); j.a_d1 = v; j.a_d2 = o;
        j.B = btov(); j.b_rows = (long long)o * v;
        j.m1_base = rz.orb0; j.m1_ext = rz.len; j.m2_ext = v;
        j.n_base = ry.orb0 * v; j.n_ext = (long long)ry.len * v;
        j.sM1 = (long long)ns * v * v; j.sM2 = v; j.sN1 = (long long)v * v; j.sN2 = 1; j.n2_ext = v;
        j.C = J() + pair0 * v * v;
        BQC_TRY(run_df_gemm(j, s));
      }
    }
  }
  return BQC_OK;
}

int Engine::exec_compute(int chunk, size_t trip0, size_t ntrip, cudaStream_t s) {
  GemmParams prm;
  memset(&prm, 0, sizeof(prm));
  prm.ntasks = (int)(3 * ntrip);
  prm.tasks = tasks_dev(chunk) + 3 * trip0;
  prm.C = F();
  if (P.profile) BQC_TRY(prof_mark(prof_main, s));
  BQC_TRY(launch_f_gemm(prm, s));
  if (P.profile) BQC_TRY(prof_mark(prof_main, s));

  EnergyArgs e;
  e.F = F(); e.trips = trips_dev(chunk) + trip0; e.orbits = orbits_dev();
  e.J = J(); e.t1 = t1p(); e.eps_occ = eps_o(); e.eps_vir = eps_v();
  e.partial = partial();
  e.t2 = in.t2; e.f_ov = fp(); e.o = P.o; e.dual = P.dual ? 1 : 0;
  e.ntrip = (int)ntrip; e.norbits = P.norbits; e.nbv = P.nbv; e.v = P.v; e.nw = P.nslots; e.use_t1 = P.use_t1;
  BQC_TRY(launch_energy(e, s));
  BQC_TRY(launch_reduce_triplets(partial(), trips_dev(chunk) + trip0, (int)ntrip, P.norbits, etrip(), s));
  if (P.profile) BQC_TRY(prof_mark(prof_main, s));
  return BQC_OK;
}

// One block triple: its triplet records and F tasks are written into the next pinned chunk, uploaded on the
// main stream (stream order protects the device chunk: its previous user, two block triples ago, ran earlier
// on the same stream), and evaluated `nbatch` triplets per W-builder launch.
int Engine::exec_triple(const Action& a, cudaStream_t s) {
  const int b = chunk_next;
  chunk_next ^= 1;
  // (while a graph is captured nothing executes: a captured schedule has at most two block triples, so each
  // pinned half is written once and stays as the replayed copies need it)
  if (!capturing && ev_up_valid[b]) BQC_CUDA_OK(cudaEventSynchronize(ev_up[b]));   // the upload that last read this half
  const size_t n = list_triple(a, trips_host(b), tasks_host(b));
  BQC_CUDA_OK(cudaMemcpyAsync(trips_dev(b), trips_host(b), n * sizeof(TripletRec), cudaMemcpyHostToDevice, s));
  BQC_CUDA_OK(cudaMemcpyAsync(tasks_dev(b), tasks_host(b), 3 * n * sizeof(GemmTask), cudaMemcpyHostToDevice, s));
  if (!capturing) {
    BQC_CUDA_OK(cudaEventRecord(ev_up[b], s));
    ev_up_valid[b] = true;
  }
  for (size_t t0 = 0; t0 < n; t0 += P.nbatch)
    BQC_TRY(exec_compute(b, t0, std::min(n - t0, (size_t)P.nbatch), s));
  return BQC_OK;
}

int Engine::execute() {
  for (const Action& a : actions) {
    if (a.kind == Action::FORM) {
      // the former stream may overwrite a slot set only after the main stream's last use of it
      if (ev_free_valid[a.set]) BQC_CUDA_OK(cudaStreamWaitEvent(s_form, ev_free[a.set], 0));
      if (P.profile) BQC_TRY(prof_mark(prof_form, s_form));
      BQC_TRY(exec_form(a.set, a.block, s_form));
      if (P.profile) BQC_TRY(prof_mark(prof_form, s_form));
      BQC_CUDA_OK(cudaEventRecord(ev_formed[a.set], s_form));
      BQC_CUDA_OK(cudaStreamWaitEvent(s_main, ev_formed[a.set], 0));
    } else if (a.kind == Action::PAIR) {
      // pair blocks are written and read on the main stream only: stream order is the only ordering needed
      if (P.profile) BQC_TRY(prof_mark(prof_form, s_main));
      BQC_TRY(exec_pair(a, s_main));
      if (P.profile) BQC_TRY(prof_mark(prof_form, s_main));
    } else {
      BQC_TRY(exec_triple(a, s_main));
      const int used[3] = {0, a.sJ, a.sK};
      for (int n = 0; n < 3; ++n) {
        BQC_CUDA_OK(cudaEventRecord(ev_free[used[n]], s_main));
        ev_free_valid[used[n]] = true;
      }
    }
  }
  // join the former stream back into the caller's stream
  BQC_CUDA_OK(cudaEventRecord(ev_join, s_form));
  BQC_CUDA_OK(cudaStreamWaitEvent(s_main, ev_join, 0));
  return BQC_OK;
}

// ------------------------------------------------------------------ one evaluation
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
  if (in.f_ov) BQC_TRY(check_device_ptr(in.f_ov, "opts->f_ov"));
  return BQC_OK;
}

int denominator_error(double emax, double vmin) {
  set_error(BQC_ERR_DENOMINATOR, "3*max(eps_occ)=%g - 3*min(eps_vir)=%g >= 0: denominators may vanish",
            3.0 * emax, 3.0 * vmin);
  return BQC_ERR_DENOMINATOR;
}

// Everything of one evaluation that is enqueued on the stream(s), from the first memset to the last sum.
int Engine::enqueue(double* e_triplet_dev, cudaStream_t stream) {
  const bool prof = P.profile != 0;
  const bool check_first = ncompute > 64;
  // esum: [0] E, [1] denominator verdict (0 ok), [2] max eps_occ, [3] min eps_vir
  BQC_CUDA_OK(cudaMemsetAsync(esum(), 0, 32, stream));
  if (!check_first) BQC_TRY(launch_denominator_check(in.eps_occ, nocc, in.eps_vir, nvir, esum() + 1, stream));
  BQC_TRY(prepare(stream));
  if (prof) BQC_CUDA_OK(cudaEventRecord(prof_prepared, stream));
  BQC_TRY(execute());
  BQC_TRY(launch_final_sum(etrip(), (long long)num_triplets(P.o), esum(), stream));
  if (prof) BQC_CUDA_OK(cudaEventRecord(prof_end, stream));
  if (e_triplet_dev)
    BQC_CUDA_OK(cudaMemcpyAsync(e_triplet_dev, etrip(), num_triplets(P.o) * 8, cudaMemcpyDeviceToDevice, stream));
  return BQC_OK;
}

int Engine::run(const Inputs& inputs, double* e_total_host, double* e_triplet_dev, cudaStream_t stream) {
  in = inputs;
  s_main = stream;
  const bool prof = P.profile != 0;
  const long long launches0 = g_launches;
  ev_used = 0;
  prof_main.clear();
  prof_form.clear();
  // Reading G10: refuse inputs whose denominators can vanish.  A long run checks before it starts (one
  // blocking 8(o+v)-byte read-back); a short one lets a kernel evaluate the bound on the stream and reads the
  // verdict together with the result, so that the call has a single host synchronisation.
  const bool check_first = ncompute > 64;
  if (check_first) {
    std::vector<double> eo(nocc), ev(nvir);
    BQC_CUDA_OK(cudaMemcpyAsync(eo.data(), in.eps_occ, (size_t)nocc * 8, cudaMemcpyDeviceToHost, stream));
    BQC_CUDA_OK(cudaMemcpyAsync(ev.data(), in.eps_vir, (size_t)nvir * 8, cudaMemcpyDeviceToHost, stream));
    BQC_CUDA_OK(cudaStreamSynchronize(stream));
    const double emax = *std::max_element(eo.begin(), eo.end());
    const double vmin = *std::min_element(ev.begin(), ev.end());
    if (!(3.0 * emax - 3.0 * vmin < 0.0)) return denominator_error(emax, vmin);
  }
  if (prof) {
    if (!prof_begin) {
      BQC_CUDA_OK(cudaEventCreate(&prof_begin));
      BQC_CUDA_OK(cudaEventCreate(&prof_prepared));
      BQC_CUDA_OK(cudaEventCreate(&prof_end));
    }
    BQC_CUDA_OK(cudaEventRecord(prof_begin, stream));
  }
  if (graph_eligible()) {
    // Short schedule: replay the captured graph when the argument pointers repeat, else (re)capture it.
    const void* key[10] = {in.eps_occ, in.eps_vir, in.t1, in.t2, in.B_oo, in.B_ov, in.B_vv, in.f_ov, e_triplet_dev,
                           this};
    if (!graph_exec || memcmp(key, graph_key, sizeof(key)) != 0) {
      if (graph_exec) { cudaGraphExecDestroy(graph_exec); graph_exec = nullptr; }
      // the pinned chunks must be quiescent before they are rewritten for the capture
      for (int b = 0; b < 2; ++b)
        if (ev_up_valid[b]) { BQC_CUDA_OK(cudaEventSynchronize(ev_up[b])); ev_up_valid[b] = false; }
      chunk_next = 0;
      cudaGraph_t graph = nullptr;
      // captured on an internal stream (the caller's may be the legacy default stream, which cannot capture);
      // the instantiated graph is launched on the caller's stream
      if (!s_cap) BQC_CUDA_OK(cudaStreamCreateWithFlags(&s_cap, cudaStreamNonBlocking));
      BQC_CUDA_OK(cudaStreamBeginCapture(s_cap, cudaStreamCaptureModeRelaxed));
      capturing = true;
      s_main = s_cap;
      const int rc = enqueue(e_triplet_dev, s_cap);
      s_main = stream;
      capturing = false;
      const cudaError_t ce = cudaStreamEndCapture(s_cap, &graph);
      if (rc != BQC_OK) {
        if (graph) cudaGraphDestroy(graph);
        cudaGetLastError();
        return rc;
      }
      BQC_CUDA_OK(ce);
      const cudaError_t ie = cudaGraphInstantiate(&graph_exec, graph, 0);
      cudaGraphDestroy(graph);
      BQC_CUDA_OK(ie);
      memcpy(graph_key, key, sizeof(key));
      graph_launches = g_launches - launches0;
    } else {
      g_launches += graph_launches;   // the replay launches the same kernels
    }
    BQC_CUDA_OK(cudaGraphLaunch(graph_exec, stream));
  } else {
    BQC_TRY(enqueue(e_triplet_dev, stream));
  }
  double res[4] = {0, 0, 0, 0};
  BQC_CUDA_OK(cudaMemcpyAsync(res, esum(), 32, cudaMemcpyDeviceToHost, stream));
  BQC_CUDA_OK(cudaStreamSynchronize(stream));   // joins s_form too (ev_join)
  g_profile[8] = (double)(g_launches - launches0);
  if (res[1] != 0.0) return denominator_error(res[2], res[3]);
  *e_total_host = res[0];
  if (prof) {
    double gemm_ms = 0, en_ms = 0, form_ms = 0;
    float ms = 0.f;
    for (size_t n = 0; n + 2 < prof_main.size() + 1; n += 3) {
      BQC_CUDA_OK(cudaEventElapsedTime(&ms, prof_main[n], prof_main[n + 1]));
      gemm_ms += ms;
      BQC_CUDA_OK(cudaEventElapsedTime(&ms, prof_main[n + 1], prof_main[n + 2]));
      en_ms += ms;
    }
    for (size_t n = 0; n + 1 < prof_form.size(); n += 2) {
      BQC_CUDA_OK(cudaEventElapsedTime(&ms, prof_form[n], prof_form[n + 1]));
      form_ms += ms;
    }
    size_t nform = 0;
    for (const Action& a : actions) nform += (a.kind == Action::FORM);
    g_profile[0] = gemm_ms;
    g_profile[1] = (double)(prof_main.size() / 3);
    g_profile[2] = en_ms;
    g_profile[3] = (double)(prof_main.size() / 3);
    g_profile[4] = form_ms;
    g_profile[5] = (double)nform;
    BQC_CUDA_OK(cudaEventElapsedTime(&ms, prof_begin, prof_prepared));
    g_profile[6] = ms;
    BQC_CUDA_OK(cudaEventElapsedTime(&ms, prof_begin, prof_end));
    g_profile[7] = ms;
  }
  return BQC_OK;
}

// ------------------------------------------------------------------ engine reuse
// The last engine of this thread is kept and reused when the next call has the same sizes, options,
// workspace and device: its streams, events, tensor maps and schedule are then not rebuilt.  An engine that
// owns its workspace is kept only while that workspace is small (kKeepBytes); bqc_release_cached() drops it.
constexpr size_t kKeepBytes = (size_t)2 << 30;
thread_local std::unique_ptr<Engine> g_engine;

bool same_opts(const bqc_t_opts& a, const bqc_t_opts* b) {
  bqc_t_opts z;
  memset(&z, 0, sizeof(z));
  if (b) z = *b;
  return a.occ_block == z.occ_block && a.occ_lo == z.occ_lo && a.occ_hi == z.occ_hi &&
         a.shard_rank == z.shard_rank && a.shard_count == z.shard_count && a.max_batch == z.max_batch &&
         a.flags == z.flags && a.workspace_gib == z.workspace_gib && (a.f_ov != nullptr) == (z.f_ov != nullptr);
}

int engine_for(int nocc, int nvir, int naux, const bqc_t_opts* opts, void* workspace, size_t workspace_bytes,
               Engine** out) {
  int dev = -1;
  BQC_CUDA_OK(cudaGetDevice(&dev));
  Engine* e = g_engine.get();
  if (e && e->nocc == nocc && e->nvir == nvir && e->naux == naux && e->device == dev && e->key_ws == workspace &&
      e->key_ws_bytes == workspace_bytes && same_opts(e->key_opts, opts)) {
    *out = e;
    return BQC_OK;
  }
  g_engine.reset();   // frees the old workspace before the new one is allocated
  std::unique_ptr<Engine> fresh(new Engine());
  BQC_TRY(fresh->init(nocc, nvir, naux, opts, workspace, workspace_bytes, nullptr));
  g_engine = std::move(fresh);
  *out = g_engine.get();
  return BQC_OK;
}

int t_energy_impl(int nocc, int nvir, int naux, const Inputs& in, const bqc_t_opts* opts, void* workspace,
                  size_t workspace_bytes, double* e_total_host, double* e_triplet_dev, cudaStream_t stream) {
  clear_error();
  if (!e_total_host) {
    set_error(BQC_ERR_NULL_POINTER, "e_total_host is NULL");
    return BQC_ERR_NULL_POINTER;
  }
  BQC_TRY(validate_inputs(nocc, nvir, naux, in));
  if (e_triplet_dev) BQC_TRY(check_device_ptr(e_triplet_dev, "e_triplet_dev"));
  const bool dual = opts && (opts->flags & BQC_T_FLAG_ABC_DRIVEN);
  const int o = dual ? nvir : nocc;   // extent of the outer index
  int lo, hi;
  BQC_TRY(resolve_window(o, opts, &lo, &hi));
  if (hi - lo < 2) {
    // a single outer orbital: only the diagonal triplet, which contributes exactly 0;
    // nocc = 1 is two electrons, no triples.  The denominator precondition (G10) is still checked.
    std::vector<double> eo(nocc), ev(nvir);
    BQC_CUDA_OK(cudaMemcpyAsync(eo.data(), in.eps_occ, (size_t)nocc * 8, cudaMemcpyDeviceToHost, stream));
    BQC_CUDA_OK(cudaMemcpyAsync(ev.data(), in.eps_vir, (size_t)nvir * 8, cudaMemcpyDeviceToHost, stream));
    if (e_triplet_dev) BQC_CUDA_OK(cudaMemsetAsync(e_triplet_dev, 0, num_triplets(o) * 8, stream));
    BQC_CUDA_OK(cudaStreamSynchronize(stream));
    const double emax = *std::max_element(eo.begin(), eo.end());
    const double vmin = *std::min_element(ev.begin(), ev.end());
    if (!(3.0 * emax - 3.0 * vmin < 0.0)) return denominator_error(emax, vmin);
    *e_total_host = 0.0;
    return BQC_OK;
  }
  Engine* e = nullptr;
  BQC_TRY(engine_for(nocc, nvir, naux, opts, workspace, workspace_bytes, &e));
  const int rc = e->run(in, e_total_host, e_triplet_dev, stream);
  if (rc != BQC_OK || (e->own_ws && e->P.total > kKeepBytes)) {
    cudaStreamSynchronize(stream);
    g_engine.reset();
  }
  return rc;
}

}  // namespace
}  // namespace bqc

// ====================================================================== C ABI
using namespace bqc;

extern "C" {

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
const char* bqc_version(void) { return "bqc_t 0.2 (sm_100a)"; }

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

void bqc_release_cached(void) { g_engine.reset(); }

int bqc_t_energy_ex(int nocc, int nvir, int naux, const double* eps_occ, const double* eps_vir,
                    const double* t1, const double* t2, const double* B_oo, const double* B_ov,
                    const double* B_vv, const bqc_t_opts* opts, void* workspace, size_t workspace_bytes,
                    double* e_total_host, double* e_triplet_dev, void* stream) {
  Inputs in = {eps_occ, eps_vir, t1, t2, B_oo, B_ov, B_vv, opts ? opts->f_ov : nullptr};
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

// ---- explicit plan handle: the engine without the thread-local cache --------------------------------------
int bqc_t_plan_create(int nocc, int nvir, int naux, const bqc_t_opts* opts, void* workspace,
                      size_t workspace_bytes, bqc_t_plan* plan_out) {
  clear_error();
  if (!plan_out) {
    set_error(BQC_ERR_NULL_POINTER, "plan_out is NULL");
    return BQC_ERR_NULL_POINTER;
  }
  *plan_out = nullptr;
  BQC_TRY(check_sizes(nocc, nvir, naux));
  BQC_TRY(check_device());
  if (workspace) BQC_TRY(check_device_ptr(workspace, "workspace"));
  std::unique_ptr<Engine> e(new Engine());
  BQC_TRY(e->init(nocc, nvir, naux, opts, workspace, workspace_bytes, nullptr));
  *plan_out = reinterpret_cast<bqc_t_plan>(e.release());
  return BQC_OK;
}

int bqc_t_plan_execute(bqc_t_plan plan, const double* eps_occ, const double* eps_vir, const double* t1,
                       const double* t2, const double* B_oo, const double* B_ov, const double* B_vv,
                       const double* f_ov, double* e_total_host, double* e_triplet_dev, void* stream) {
  clear_error();
  Engine* e = reinterpret_cast<Engine*>(plan);
  if (!e || !e_total_host) {
    set_error(BQC_ERR_NULL_POINTER, "%s is NULL", e ? "e_total_host" : "plan");
    return BQC_ERR_NULL_POINTER;
  }
  int dev = -1;
  BQC_CUDA_OK(cudaGetDevice(&dev));
  if (dev != e->device) {
    set_error(BQC_ERR_DEVICE, "plan was created on device %d, current device is %d", e->device, dev);
    return BQC_ERR_DEVICE;
  }
  if ((f_ov != nullptr) != (e->P.fock != 0)) {
    set_error(BQC_ERR_INVALID_OPTION, "f_ov %s but the plan was created %s opts->f_ov", f_ov ? "given" : "NULL",
              e->P.fock ? "with" : "without");
    return BQC_ERR_INVALID_OPTION;
  }
  Inputs in = {eps_occ, eps_vir, t1, t2, B_oo, B_ov, B_vv, f_ov};
  BQC_TRY(validate_inputs(e->nocc, e->nvir, e->naux, in));
  if (e_triplet_dev) BQC_TRY(check_device_ptr(e_triplet_dev, "e_triplet_dev"));
  if (e->P.na < 2) {
    set_error(BQC_ERR_INVALID_OPTION, "plan over a single outer orbital has no triplets; use bqc_t_energy_ex");
    return BQC_ERR_INVALID_OPTION;
  }
  return e->run(in, e_total_host, e_triplet_dev, static_cast<cudaStream_t>(stream));
}

void bqc_t_plan_destroy(bqc_t_plan plan) { delete reinterpret_cast<Engine*>(plan); }

size_t bqc_t_plan_workspace_bytes(bqc_t_plan plan) {
  return plan ? reinterpret_cast<Engine*>(plan)->P.total : 0;
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
  // never read.  The abc-driven schedule reads t2[:,:,a,b] for the virtuals of its window: the whole array.
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

// ---- single steps (parity tests): a private engine over the orbitals involved, one block --------------------
static int debug_engine(Engine& e, int nocc, int nvir, int naux, const Inputs& in, const std::vector<int>& act,
                        cudaStream_t stream) {
  bqc_t_opts o2;
  memset(&o2, 0, sizeof(o2));
  o2.max_batch = 1;
  o2.occ_block = (int)act.size();
  BQC_TRY(e.init(nocc, nvir, naux, &o2, nullptr, 0, &act));
  e.in = in;
  e.s_main = stream;
  BQC_TRY(e.prepare(stream));
  return BQC_OK;
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
  if (I_dev) BQC_TRY(check_device_ptr(I_dev, "I_dev"));
  if (O_dev) BQC_TRY(check_device_ptr(O_dev, "O_dev"));
  if (J_dev) BQC_TRY(check_device_ptr(J_dev, "J_dev"));
  Inputs in = {nullptr, nullptr, nullptr, t2, B_oo, B_ov, B_vv};
  std::vector<int> act;
  act.push_back(std::min(x, y));
  if (x != y) act.push_back(std::max(x, y));
  Engine e;
  BQC_TRY(debug_engine(e, nocc, nvir, naux, in, act, stream));
  const Plan& P = e.P;
  const int px = (int)(std::find(act.begin(), act.end(), x) - act.begin());
  const int py = (int)(std::find(act.begin(), act.end(), y) - act.begin());
  const int v = nvir;
  if (I_dev) {
    BQC_TRY(e.exec_form(0, 0, stream));   // one block holds all active orbitals: slot = position
    BQC_TRY(launch_copy3(e.slabs() + (size_t)px * P.slab_elems, (long long)v * P.Kp, P.Kp, 1, I_dev, v, v, v,
                         stream));
  }
  if (O_dev || J_dev) {
    Action a;
    memset(&a, 0, sizeof(a));
    a.kind = Action::PAIR;
    a.need_j = 1; a.need_panel = 1;
    BQC_TRY(e.exec_pair(a, stream));
  }
  if (O_dev)   // O_xy[l,u] = (x u|y l) = B~_xy[u, v + l]  -> out[l][u]
    BQC_TRY(launch_copy3(e.btil() + ((size_t)px * P.nslots + py) * v * P.Kp + v, 0, 1, P.Kp, O_dev, 1, nocc, v,
                         stream));
  if (J_dev)
    BQC_CUDA_OK(cudaMemcpyAsync(J_dev, e.J() + ((size_t)px * P.nslots + py) * v * v, (size_t)v * v * 8,
                                cudaMemcpyDeviceToDevice, stream));
  BQC_CUDA_OK(cudaStreamSynchronize(stream));
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
  if (i < 0 || j < 0 || k < 0 || i >= nocc || j >= nocc || k >= nocc) {
    set_error(BQC_ERR_INVALID_SIZE, "triplet (%d,%d,%d) outside [0,%d)", i, j, k, nocc);
    return BQC_ERR_INVALID_SIZE;
  }
  if (W_dev) BQC_TRY(check_device_ptr(W_dev, "W_dev"));
  if (V_dev) BQC_TRY(check_device_ptr(V_dev, "V_dev"));
  std::vector<int> act = {i, j, k};
  std::sort(act.begin(), act.end());
  act.erase(std::unique(act.begin(), act.end()), act.end());
  Engine e;
  BQC_TRY(debug_engine(e, nocc, nvir, naux, in, act, stream));
  const Plan& P = e.P;
  // the three F tasks of (i,j,k) in the caller's order (one block: slot = position in `act`)
  auto pos = [&](int x) { return (int)(std::find(act.begin(), act.end(), x) - act.begin()); };
  const int pi = pos(i), pj = pos(j), pk = pos(k);
  std::vector<GemmTask> ft;
  {
    auto pair = [&](int pz, int py) { return pz * P.nslots + py; };
    auto f_task = [&](int px, int py, int pz, int cls) {
      GemmTask g;
      memset(&g, 0, sizeof(g));
      g.nterms = 2;
      g.term[0].a_idx = px; g.term[0].a_transposed = 0; g.term[0].b_idx = pair(pz, py);
      g.term[1].a_idx = py; g.term[1].a_transposed = 1; g.term[1].b_idx = pair(pz, px);
      g.c_off = (long long)(cls * P.fsz);
      ft.push_back(g);
    };
    f_task(pi, pj, pk, 0);
    f_task(pi, pk, pj, 1);
    f_task(pj, pk, pi, 2);
  }
  // the engine's own schedule is not executed here: the three tasks go into chunk 0
  BQC_CUDA_OK(cudaMemcpyAsync(e.tasks_dev(0), ft.data(), 3 * sizeof(GemmTask), cudaMemcpyHostToDevice, stream));
  BQC_TRY(e.exec_form(0, 0, stream));
  Action a;
  memset(&a, 0, sizeof(a));
  a.kind = Action::PAIR;
  a.need_j = 1; a.need_panel = 1;
  BQC_TRY(e.exec_pair(a, stream));
  GemmParams prm;
  memset(&prm, 0, sizeof(prm));
  prm.ntasks = 3;
  prm.tasks = e.tasks_dev(0);
  prm.C = e.F();
  BQC_TRY(e.launch_f_gemm(prm, stream));
  BQC_TRY(launch_assemble_wv(e.F(), P.nbv, nvir, e.J(), P.nslots, pi, pj, pk, t1 + (size_t)i * nvir,
                             t1 + (size_t)j * nvir, t1 + (size_t)k * nvir, t2, nocc, i, j, k, f_ov, W_dev, V_dev,
                             stream));
  BQC_CUDA_OK(cudaStreamSynchronize(stream));   // `ft` and the engine go out of scope
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
    prm.ktail8 = (K - (prm.kiters - 1) * kBK) <= 8;   // TMA zero-fills beyond K
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
