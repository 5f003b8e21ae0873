// plan.cuh — sizes, workspace layout and the block-triple deal of one (T) evaluation (SURVEY.md §8(a) row a5,
// §8(e)).  Host-only logic: everything here runs without a GPU (bqc_t_workspace_bytes, bqc_t_flops, ...).
//
// "Pipeline space": the scheduler always walks triplets x <= y <= z of an OUTER index of extent `o` with all
// `v`^3 INNER index triples inside.  For the ijk-driven schedule outer = occupied, inner = virtual; for the
// abc-driven schedule (BQC_T_FLAG_ABC_DRIVEN) the two swap roles (particle-hole duality,
// DESIGN.md §11) and Plan::dual is set: o = nvir, v = nocc.
#pragma once

#include <vector>

#include "common.cuh"

namespace bqc {

struct Plan {
  int o = 0, v = 0, X = 0;     // pipeline-space extents (see above)
  bool dual = false;           // abc-driven: outer index = the caller's virtual orbitals
  std::vector<int> act;        // active outer orbitals (sorted); triplets are drawn from these
  int na = 0;                  // act.size()
  int Xp = 0, Kp = 0;          // aux / (v+o) extents padded to multiples of 16
  int nbv = 0;                 // 8-blocks per inner dimension
  size_t fsz = 0;              // doubles per blocked F array
  size_t slab_elems = 0;       // v*v*Kp
  int Bo = 0, nblk = 0, nsets = 0, nslots = 0;
  int nbatch = 0;              // triplets per W-builder launch
  int norbits = 0;
  int nruns = 1;               // contiguous runs in `act`
  int use_t1 = 1;
  int profile = 0;
  int fock = 0;                // opts->f_ov given
  int shard_rank = 0, shard_count = 1;
  int shard_blocks = 0;        // BQC_T_FLAG_SHARD_BLOCKS
  // workspace offsets (bytes)
  size_t off_btvv = 0, off_btov = 0, off_panel = 0, off_btil = 0, off_J = 0, off_slabs = 0, off_F = 0,
         off_partial = 0, off_etrip = 0, off_esum = 0, off_act = 0, off_orbits = 0, off_tasks = 0,
         off_trips = 0, off_small = 0, total = 0;
  size_t small_eo = 0, small_ev = 0, small_t1 = 0, small_f = 0;   // dual copies of eps/t1/f inside off_small
  size_t chunk_trips = 0;      // triplets per schedule chunk (the largest block triple)
  // names + sizes of the largest buffers, for BQC_ERR_WORKSPACE details
  const char* biggest_name = "";
  size_t biggest_bytes = 0;
};

size_t num_triplets(int o);
// lexicographic rank of (i,j,k), i <= j <= k < o
size_t triplet_index(int o, int i, int j, int k);

// Resolve the window [lo,hi) of the outer index from opts (occ_lo = occ_hi = 0: everything).
int resolve_window(int o, const bqc_t_opts* opts, int* lo, int* hi);

// Fill every field of P for outer extent o, inner extent v (pipeline space) and active list `act`.
int make_plan(Plan& P, int o, int v, int X, bool dual, const std::vector<int>& act, const bqc_t_opts* opts);

// Plan of a caller-space problem: handles BQC_T_FLAG_ABC_DRIVEN (swaps o and v) and the window.
int make_plan_for(Plan& P, int nocc, int nvir, int naux, const bqc_t_opts* opts);

// Non-diagonal triplets pi <= pj <= pk of block triple (I, J, K) over na orbitals in blocks of bo.
long long block_triple_work(int na, int bo, int I, int J, int K);

// BQC_T_FLAG_SHARD_BLOCKS: owner of every block triple I <= J <= K (numbered in loop order).  Largest block
// triples first, each to the least-loaded rank so far (ties: lower rank) — a deterministic function of
// (na, bo, shard_count), so every rank and the host helpers (bqc_t_flops, bqc_t_triplet_owner_ex) agree.
std::vector<int> deal_block_triples(int na, int bo, int shard_count, std::vector<long long>* load_out = nullptr);

}  // namespace bqc
