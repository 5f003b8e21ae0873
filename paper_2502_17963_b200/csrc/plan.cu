// plan.cu — host-only planning: workspace layout, block sizes from a memory budget, the block-triple deal of
// the multi-GPU path, and the host-only entry points of the C ABI that follow from them.
#include "plan.cuh"

#include <math.h>
#include <string.h>

#include <algorithm>

#include "gemm_nt.cuh"
#include "kernels.cuh"

namespace bqc {

size_t num_triplets(int o) { return (size_t)o * (o + 1) * (o + 2) / 6; }

size_t triplet_index(int o, int i, int j, int k) {
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
    set_error(BQC_ERR_INVALID_OPTION, "window [%d,%d) invalid for an outer extent of %d", *lo, *hi, o);
    return BQC_ERR_INVALID_OPTION;
  }
  return BQC_OK;
}

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

std::vector<int> deal_block_triples(int na, int bo, int shard_count, std::vector<long long>* load_out) {
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

namespace {

// Block size for a block-triple-sharded run: the largest Bo <= the memory-derived one whose deal is within
// 3 % of even (the slabs of a block are re-formed by every rank that owns one of its triples, so larger is
// cheaper); the best one found if none is.
int balanced_block(int na, int bo_max, int shard_count) {
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

constexpr double kGiB = 1073741824.0;

}  // namespace

int make_plan(Plan& P, int o, int v, int X, bool dual, const std::vector<int>& act, const bqc_t_opts* opts) {
  P.o = o; P.v = v; P.X = X; P.dual = dual;
  P.act = act;
  P.na = (int)act.size();
  P.nruns = 1;
  for (int p = 1; p < P.na; ++p)
    if (act[p] != act[p - 1] + 1) ++P.nruns;
  P.Xp = round_up_i(X, 16);
  P.Kp = round_up_i(v + o, 16);
  P.nbv = ceil_div(v, kVB);
  P.fsz = (size_t)P.nbv * P.nbv * P.nbv * (kVB * kVB * kVB);
  P.slab_elems = (size_t)v * v * P.Kp;
  P.norbits = (int)((long long)P.nbv * (P.nbv + 1) * (P.nbv + 2) / 6);
  P.use_t1 = !(opts && (opts->flags & BQC_T_FLAG_NO_T1));
  P.profile = (opts && (opts->flags & BQC_T_FLAG_PROFILE)) ? 1 : 0;
  P.fock = (opts && opts->f_ov) ? 1 : 0;
  P.shard_count = (opts && opts->shard_count > 0) ? opts->shard_count : 1;
  P.shard_rank = opts ? opts->shard_rank : 0;
  P.shard_blocks = (opts && (opts->flags & BQC_T_FLAG_SHARD_BLOCKS)) ? 1 : 0;
  if (P.shard_rank < 0 || P.shard_rank >= P.shard_count) {
    set_error(BQC_ERR_INVALID_OPTION, "shard_rank %d outside [0,%d)", P.shard_rank, P.shard_count);
    return BQC_ERR_INVALID_OPTION;
  }
  const int bo_opt = opts ? opts->occ_block : 0;
  const int gib_opt = opts ? opts->workspace_gib : 0;
  if (bo_opt < 0 || gib_opt < 0) {
    set_error(BQC_ERR_INVALID_OPTION, "occ_block %d / workspace_gib %d < 0", bo_opt, gib_opt);
    return BQC_ERR_INVALID_OPTION;
  }
  // Budget for the buffers whose size follows the block size: 2/3 for the 4 slab sets, 1/3 for the 16
  // set-pair blocks of B~ and J.  A single block (everything resident once) is taken when it fits.
  const double budget = (gib_opt > 0 ? (double)gib_opt : 36.0) * kGiB;
  const double slab_bytes = (double)P.slab_elems * 8.0;
  const double pair_bytes = ((double)v * P.Kp + (double)v * v) * 8.0;
  if (bo_opt > 0) {
    P.Bo = std::min(bo_opt, P.na);
  } else if (P.na * slab_bytes <= budget * (2.0 / 3.0) && (double)P.na * P.na * pair_bytes <= budget / 3.0) {
    P.Bo = P.na;
  } else {
    const int bo_slab = (int)floor(budget * (2.0 / 3.0) / (4.0 * slab_bytes));
    const int bo_pair = (int)floor(sqrt(budget / 3.0 / (16.0 * pair_bytes)));
    int bo = std::max(1, std::min(std::min(bo_slab, bo_pair), P.na));
    bo = ceil_div(P.na, ceil_div(P.na, bo));   // balanced blocks
    P.Bo = bo;
  }
  if (bo_opt == 0 && P.shard_blocks && P.shard_count > 1) P.Bo = balanced_block(P.na, P.Bo, P.shard_count);
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
    nbatch = (int)floor(6.0 * kGiB / per);
  }
  P.nbatch = std::max(1, std::min(nbatch, 1024));

  // The schedule reaches the device one block triple at a time, into one of two chunks: a chunk holds the
  // triplet records and F-GEMM tasks of the largest block triple (all of them when there is one block).
  const size_t ntrip_act = (size_t)P.na * (P.na + 1) * (P.na + 2) / 6;
  P.chunk_trips = P.nblk == 1 ? ntrip_act : std::min(ntrip_act, (size_t)P.Bo * P.Bo * P.Bo);

  size_t off = 0;
  P.biggest_bytes = 0;
  auto take = [&](size_t bytes, const char* name) {
    size_t r = off;
    off = round_up(off + bytes, 1024);
    if (bytes > P.biggest_bytes) { P.biggest_bytes = bytes; P.biggest_name = name; }
    return r;
  };
  P.off_btvv = take((size_t)v * v * P.Xp * 8, "K-major copy of the inner-inner DF block [v*v][Xp]");
  P.off_btov = take((size_t)o * v * P.Xp * 8, "K-major copy of B_ov [o*v][Xp]");
  P.off_panel = take((size_t)P.Bo * o * P.Xp * 8, "K-major panel of the outer-outer DF block [Bo*o][Xp]");
  P.off_btil = take((size_t)P.nslots * P.nslots * v * P.Kp * 8, "B~ pair blocks [nslots^2][v][Kp]");
  P.off_J = take((size_t)P.nslots * P.nslots * v * v * 8, "J pair blocks [nslots^2][v][v]");
  P.off_slabs = take((size_t)P.nslots * P.slab_elems * 8, "augmented slab cache [nslots][v][v][Kp]");
  P.off_F = take((size_t)P.nbatch * 3 * P.fsz * 8, "F arrays of one batch [nbatch][3][v^3]");
  P.off_partial = take((size_t)P.nbatch * P.norbits * 8, "per-orbit partial sums");
  P.off_etrip = take(num_triplets(o) * 8, "per-triplet energies");
  P.off_esum = take(64, "result");
  P.off_act = take((size_t)P.na * 4, "active list");
  P.off_orbits = take((size_t)P.norbits * 4, "orbit table");
  P.off_tasks = take((8 + 2 * 3 * P.chunk_trips) * sizeof(GemmTask), "GEMM task chunks");
  P.off_trips = take(2 * P.chunk_trips * sizeof(TripletRec), "triplet record chunks");
  {
    // dual copies of the small inputs (abc-driven schedule): eps_occ', eps_vir', t1', f'
    size_t s = 0;
    auto sub = [&](size_t bytes) { size_t r = s; s = round_up(s + bytes, 256); return r; };
    P.small_eo = sub((size_t)o * 8);
    P.small_ev = sub((size_t)v * 8);
    P.small_t1 = sub((size_t)o * v * 8);
    P.small_f = sub((size_t)o * v * 8);
    P.off_small = take(dual ? s : 0, "dual copies of eps/t1/f");
  }
  P.total = off;
  return BQC_OK;
}

int make_plan_for(Plan& P, int nocc, int nvir, int naux, const bqc_t_opts* opts) {
  const bool dual = opts && (opts->flags & BQC_T_FLAG_ABC_DRIVEN);
  const int o = dual ? nvir : nocc, v = dual ? nocc : nvir;
  int lo, hi;
  BQC_TRY(resolve_window(o, opts, &lo, &hi));
  std::vector<int> act(hi - lo);
  for (int x = lo; x < hi; ++x) act[x - lo] = x;
  return make_plan(P, o, v, naux, dual, act, opts);
}

}  // namespace bqc

// ====================================================================== host-only C ABI
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
  bqc_t_opts o2;
  memset(&o2, 0, sizeof(o2));
  if (opts) o2 = *opts;
  o2.shard_rank = 0;
  Plan P;
  if (make_plan_for(P, nocc, nvir, naux, &o2) != BQC_OK) return -1;
  const int lo = P.act.front(), hi = P.act.back() + 1;
  if (i < lo || i > j || j > k || k >= hi) return -1;
  if (!P.shard_blocks) return (int)(triplet_index(P.o, i, j, k) % (size_t)P.shard_count);
  // block triples I <= J <= K are numbered in loop order = lexicographic rank among the nblk blocks
  const size_t bt = triplet_index(P.nblk, (i - lo) / P.Bo, (j - lo) / P.Bo, (k - lo) / P.Bo);
  return deal_block_triples(P.na, P.Bo, P.shard_count)[bt];
}

double bqc_t_flops(int nocc, int nvir, const bqc_t_opts* opts) {
  clear_error();
  if (nocc <= 0 || nvir <= 0) return 0.0;
  Plan P;
  if (make_plan_for(P, nocc, nvir, 1, opts) != BQC_OK) return -1.0;
  size_t n = 0;
  if (P.shard_blocks && P.shard_count > 1) {
    std::vector<long long> load;
    deal_block_triples(P.na, P.Bo, P.shard_count, &load);
    n = (size_t)load[P.shard_rank];
  } else {
    for (int i : P.act)
      for (int j = i; j <= P.act.back(); ++j)
        for (int k = j; k <= P.act.back(); ++k) {
          if (i == j && j == k) continue;
          if ((int)(triplet_index(P.o, i, j, k) % (size_t)P.shard_count) == P.shard_rank) ++n;
        }
  }
  const double v = P.v;   // pipeline space: 12 v^3 (v + o) per outer triplet (12 o^3 (v+o) per virtual triple)
  return (double)n * 12.0 * v * v * v * (v + P.o);
}

int bqc_t_plan_occ_block(int nocc, int nvir, int naux, const bqc_t_opts* opts) {
  clear_error();
  if (check_sizes(nocc, nvir, naux) != BQC_OK) return -1;
  Plan P;
  if (make_plan_for(P, nocc, nvir, naux, opts) != BQC_OK) return -1;
  return P.Bo;
}

size_t bqc_t_workspace_bytes(int nocc, int nvir, int naux, const bqc_t_opts* opts) {
  clear_error();
  if (check_sizes(nocc, nvir, naux) != BQC_OK) return 0;
  Plan P;
  if (make_plan_for(P, nocc, nvir, naux, opts) != BQC_OK) return 0;
  return P.total;
}

}  // extern "C"
