// gemm_nt.cuh — the one FP64 tile-GEMM engine of the library.
//
//   C[(m1,m2), n] = sum_terms sum_k A_term[(m1,m2), k] * B_term[n, k]           ("NT", both K-major)
//
// * Operands are staged global -> shared by TMA (cp.async.bulk.tensor, 128-byte swizzle) through a
//   ring of mbarrier-guarded stages filled by one producer warp.
// * 8 consumer warps issue FP64 tensor-core MMAs (mma.sync m8n8k4 -> SASS DMMA.8x8x4; sm_100a has no
//   tcgen05/wgmma f64 kind) on a 128 x 128 CTA tile, 64 x 32 per warp, accumulators in registers.
// * Blocked (F-layout) output leaves through shared memory: the consumers write their accumulators into a
//   staging tile (each fragment block is one contiguous 512-byte run of the 8^3-blocked layout) and go
//   straight on to the next tile, while a "store warp" drains the staging tile to global memory with bulk
//   async copies (cp.async.bulk shared -> global).  Measured: direct st.global from the consumers costs
//   3.6 us per 128 KB tile (7 % of a config-3 step) because the stores back up the LSU/MIO queues that the
//   fragment ld.shared of the main loop also need; the staged epilogue costs the st.shared time only.
// * The kernel is persistent: CTAs stride over a tile list ordered (m1-tile, m2-tile, task, n-tile), n fastest,
//   so that concurrently running CTAs share the A tile through L2 — across the column tiles of a task and
//   across the tasks of a launch that read the same slab.
// * The M index is a pair (m1, m2) tiled tp x tq (tp*tq = 128).  A term may read its A rows from the
//   same tensor with (m1, m2) transposed ("a_transposed": tp single-row-block TMA boxes instead of
//   one), which is how W's index-permuted slab reads (I_y[q,p,:]) cost nothing.
#pragma once

#include <type_traits>

#include "common.cuh"

namespace bqc {

constexpr int kBM = 128;            // rows of the A tile (= tp * tq)
constexpr int kBK = 16;             // doubles per smem row = 128 bytes = one swizzle span
constexpr int kConsumerWarps = 8;   // 4 (M) x 2 (N) warps, warp tile 32 x (8*NF0 | 8*NF1)
constexpr int kGemmThreads = (kConsumerWarps + 4) * 32;   // 2 consumer warpgroups + 1 producer/store warpgroup
// The B tile has BN = 8*NF rows: NF 8-column MMA fragments, NF0 = ceil(NF/2) owned by warp column 0 and
// NF1 = floor(NF/2) by warp column 1 (odd NF: the last fragment of column 1 is switched off), NF in
// [kMinNF, kMaxNF].  So any N extent is covered to within 8 columns.
constexpr int kMinNF = 4, kMaxNF = 16;
#ifdef __CUDACC__
#define BQC_HD __host__ __device__
#else
#define BQC_HD
#endif
constexpr int kSmemBudget = 227 * 1024;   // dynamic shared memory per CTA on sm_100
BQC_HD constexpr int gemm_bn(int nf) { return 8 * nf; }
BQC_HD constexpr int gemm_stage_bytes(int nf) { return (kBM + gemm_bn(nf)) * kBK * 8; }
// staging tile of the blocked-output epilogue: the whole 128 x 8*NF accumulator tile
BQC_HD constexpr int gemm_staging_bytes(int nf, bool staged) { return staged ? kBM * gemm_bn(nf) * 8 : 0; }
BQC_HD constexpr int gemm_stages(int nf, bool staged) {
  return (kSmemBudget - 1024 - 256 - gemm_staging_bytes(nf, staged)) / gemm_stage_bytes(nf) > 6
             ? 6
             : (kSmemBudget - 1024 - 256 - gemm_staging_bytes(nf, staged)) / gemm_stage_bytes(nf);
}
BQC_HD constexpr int gemm_smem_bytes(int nf, bool staged) {
  return gemm_stages(nf, staged) * gemm_stage_bytes(nf) + gemm_staging_bytes(nf, staged) + 1024 /*align slack*/ +
         256 /*barriers*/;
}

struct GemmTerm {
  int a_idx;          // coordinate 3 of the A tensor map (slab slot / batch entry)
  int b_idx;          // coordinate 2 of the B tensor map (pair index / batch entry)
  int a_transposed;   // 0: A row (m1,m2) = tensor[a_idx][m1][m2][:]; 1: = tensor[a_idx][m2][m1][:]
  int pad;
};

struct GemmTask {
  GemmTerm term[2];
  long long c_off;    // element offset of this task's output inside C
  int nterms;
  int pad;
};

struct GemmParams {
  int ntasks;
  int tiles_m1, tiles_m2, tiles_n;   // per task
  int tp, tq_log2;                   // M tile = tp (m1) x tq (m2), tq = 1 << tq_log2
  int m1_base, n_base;               // added to the TMA coordinates (not to the output index)
  int m1_out, n_out;                 // added to the output index (a launch may cover a sub-range of M1 / N)
  int m1_ext, m2_ext, n_ext;         // valid extents of the output index ranges
  int kiters;                        // ceil(K / 16) per term
  int ktail8;                        // 1: the last stage of every term holds <= 8 valid K columns: selects the kTail
                                     //    instantiation, whose last stage runs 2 of the 4 k4-steps (see gemm_consume)
  // output addressing
  int out_mode;                      // 0: strided, 1: blocked 8^3 tiles (F layout)
  int n2_ext;                        // strided: n -> (n / n2_ext, n % n2_ext)
  long long sM1, sM2, sN1, sN2;      // strided: off = c_off + m1*sM1 + m2*sM2 + n1*sN1 + n2*sN2
  int nbv;                           // blocked: 8-blocks per dimension
  const GemmTask* tasks;
  double* C;
};

#ifdef __CUDACC__

// b[J..N-1] = B fragment values of one k4 step (rows g + 8j of this warp's column half).
template <int J, int N>
__device__ __forceinline__ void load_b_frags(double (&b)[N], uint32_t pb) {
  if constexpr (J < N) {
    b[J] = lds_f64<J * 1024>(pb);
    load_b_frags<J + 1, N>(b, pb);
  }
}

// Tile number -> (task, m1-tile, m2-tile, n-tile).  n runs fastest, then the TASK, then the row tile: the tiles
// that run concurrently are the column tiles of all tasks of a launch for a few row tiles, so tasks that read the
// same slab in the same orientation (F(i,j,k) and F(i,k,j) both start from I~_i; consecutive triplets of a
// batch share I~_i and I~_j) find its A tile in L2 instead of streaming the 554 MB slab from HBM once per task.
struct TileCoord { int task_id, m1_t, m2_t, n_t; };
__device__ __forceinline__ TileCoord decode_tile(const GemmParams& prm, long long tile) {
  TileCoord c;   // 32-bit arithmetic: launch_gemm_nt refuses launches of 2^31 tiles or more
  const unsigned t = (unsigned)tile;
  const unsigned r = t / (unsigned)prm.tiles_n;
  c.n_t = (int)(t - r * (unsigned)prm.tiles_n);
  const unsigned r2 = r / (unsigned)prm.ntasks;
  c.task_id = (int)(r - r2 * (unsigned)prm.ntasks);
  c.m1_t = (int)(r2 / (unsigned)prm.tiles_m2);
  c.m2_t = (int)(r2 - (unsigned)c.m1_t * (unsigned)prm.tiles_m2);
  return c;
}

// The consumer loop of one warp that owns NFW 8-column fragments starting at tile column warp_n0.
template <int NF, int NFW, bool kStaged, bool kTail>
__device__ __forceinline__ void gemm_consume(const GemmParams& prm, uint8_t* smem, uint64_t* full_bar,
                                             uint64_t* empty_bar, uint64_t* c_full, uint64_t* c_empty,
                                             double* staging, int warp, int lane, int warp_n0,
                                             long long total_tiles, int tiles_per_task, int tq) {
  constexpr int kBN = gemm_bn(NF);
  constexpr int kStageBytes = gemm_stage_bytes(NF);
  constexpr int kStages = gemm_stages(NF, kStaged);
  uint32_t c_phase = 0;   // parity of the staging-tile hand-over (staged epilogue)
  const int g = lane >> 2;            // fragment row (A) / column (B)
  const int t = lane & 3;             // fragment k index
  const int warp_m0 = (warp & 3) * 32;
  // k slot of lane t in k4-step c is k = 2c + (t&1) + 8*(t>>1): with the 128B swizzle (16-byte chunk
  // index ^= row & 7) the 16 lanes of a half-warp then hit 16 distinct 8-byte bank pairs.
  uint32_t koff[4];
#pragma unroll
  for (int c = 0; c < 4; ++c) koff[c] = (uint32_t)((((c + 4 * (t >> 1)) ^ g) << 4) + ((t & 1) << 3));
  // K tail: when the last stage of a term holds <= 8 valid columns (prm.ktail8), that stage runs two k4-steps over
  // k = 4c + t (columns 0..7) instead of four over all 16 — the other half would only multiply TMA's zero fill.
  // This contiguous map costs a 2-way bank conflict, on that one stage only.
  uint32_t kofft[2];
#pragma unroll
  for (int c = 0; c < 2; ++c) kofft[c] = (uint32_t)((((2 * c + (t >> 1)) ^ g) << 4) + ((t & 1) << 3));
  const uint32_t smem_base = smem_u32(smem);
  const uint32_t a_base = smem_base + (uint32_t)((warp_m0 + g) * (kBK * 8));
  const uint32_t b_base = smem_base + (uint32_t)(kBM * kBK * 8 + (warp_n0 + g) * (kBK * 8));

  // fragments of one k4 step: 4 A values (rows g + 8i) and NF B values (rows g + 8j), plain ld.shared
  auto load_frags = [&](double (&a)[4], double (&b)[NFW], int stg, uint32_t kof) {
    const uint32_t off = (uint32_t)(stg * kStageBytes) + kof;
    const uint32_t pa = a_base + off, pb = b_base + off;
    a[0] = lds_f64<0 * 1024>(pa); a[1] = lds_f64<1 * 1024>(pa);
    a[2] = lds_f64<2 * 1024>(pa); a[3] = lds_f64<3 * 1024>(pa);
    load_b_frags<0, NFW>(b, pb);
  };

  int stage = 0;
  uint32_t phase = 0;
  for (long long tile = blockIdx.x; tile < total_tiles; tile += gridDim.x) {
    const TileCoord tc = decode_tile(prm, tile);
    const int task_id = tc.task_id, n_t = tc.n_t, m2_t = tc.m2_t, m1_t = tc.m1_t;
    const GemmTask* task = prm.tasks + task_id;
    const int iters = task->nterms * prm.kiters;

    double acc[4][NFW][2];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
      for (int j = 0; j < NFW; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

    // Fragments are double-buffered in registers across k4 steps AND across pipeline stages: the loads
    // of step s+1 (possibly the first step of the next stage, after its full barrier) are issued before
    // the 4*NF DMMAs of step s, so ld.shared latency and the barrier poll hide behind tensor work.
    double fa[2][4], fb[2][NFW];
    // One pipeline stage of NV k4-steps (NV = 4: a full 16-column stage; NV = 2: the short last stage of a term,
    // kTail only).  NV is even so that the next stage's first fragments always land in register buffer 0.  The
    // stage bodies are peeled below so that no stage carries a run-time test: whether a stage has a successor
    // and which k map the successor's first fragments use is fixed by its position.
    auto run_stage = [&](auto NVc, bool has_next, uint32_t next_kof) {
      constexpr int NV = decltype(NVc)::value;
      static_assert(NV == 2 || NV == 4, "even step counts only");
      int nstage = stage + 1;
      uint32_t nphase = phase;
      if (nstage == kStages) { nstage = 0; nphase ^= 1u; }
#pragma unroll
      for (int c = 0; c < NV; ++c) {
        const int cur = c & 1, nxt = cur ^ 1;
        if (c < NV - 1) {
          load_frags(fa[nxt], fb[nxt], stage, NV == 4 ? koff[(c + 1) & 3] : kofft[(c + 1) & 1]);
        } else if (has_next) {
          mbar_wait(&full_bar[nstage], nphase);
          load_frags(fa[nxt], fb[nxt], nstage, next_kof);
        }
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
          for (int j = 0; j < NFW; ++j) dmma_884(acc[i][j][0], acc[i][j][1], fa[cur][i], fb[cur][j]);
      }
      // every ld.shared of this stage was issued (and its value consumed by a DMMA above) -> release it
      __syncwarp();
      if (lane == 0) mbar_arrive(&empty_bar[stage]);
      stage = nstage;
      phase = nphase;
    };
    if constexpr (!kTail) {
      mbar_wait(&full_bar[stage], phase);
      load_frags(fa[0], fb[0], stage, koff[0]);
      for (int it = 0; it + 1 < iters; ++it) run_stage(std::integral_constant<int, 4>{}, true, koff[0]);
      run_stage(std::integral_constant<int, 4>{}, false, 0u);
    } else {
      // every term is (kiters - 1) full stages + one short stage of two k4-steps
      const int kfull = prm.kiters - 1;
      mbar_wait(&full_bar[stage], phase);
      load_frags(fa[0], fb[0], stage, kfull > 0 ? koff[0] : kofft[0]);
      const int nterms = task->nterms;
      for (int term = 0; term < nterms; ++term) {
        for (int s = 0; s + 1 < kfull; ++s) run_stage(std::integral_constant<int, 4>{}, true, koff[0]);
        if (kfull > 0) run_stage(std::integral_constant<int, 4>{}, true, kofft[0]);      // the next stage is short
        run_stage(std::integral_constant<int, 2>{}, term + 1 < nterms, kfull > 0 ? koff[0] : kofft[0]);
      }
    }

    if constexpr (kStaged) {
      // ------------------------- epilogue: registers -> staging tile -> (store warp) -------------------------
      // Fragment block (i, j) of this warp — rows warp_m0 + 8i + g, columns warp_n0 + 8j + 2t, +1 — is one
      // 8 x 8 block of the 8^3-blocked F layout for a fixed m1 (tq >= 8): a contiguous 512-byte run, written
      // by one conflict-free warp-wide 16-byte store.  Run index = (row group, column block).
      mbar_wait(c_empty, c_phase ^ 1u);          // the store warp has read the previous tile out of staging
      const uint32_t st = smem_u32(staging) +
                          (uint32_t)(((((warp_m0 >> 3) * (kBN >> 3) + (warp_n0 >> 3)) << 6) + (g << 3) + 2 * t) << 3);
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < NFW; ++j)
          sts_v2_f64(st + (uint32_t)((i * (kBN >> 3) + j) << 9), acc[i][j][0], acc[i][j][1]);
      fence_proxy_async();                       // generic-proxy writes -> visible to the bulk-copy engine
      __syncwarp();
      if (lane == 0) mbar_arrive(c_full);
      c_phase ^= 1u;
      continue;
    }
    // ------------------------------- epilogue: registers -> global -------------------------------
    const int m1_0 = prm.m1_out + m1_t * prm.tp;
    const int m2_0 = m2_t * tq;
    const int n_0 = prm.n_out + n_t * kBN + warp_n0 + 2 * t;
    double* __restrict__ C = prm.C + task->c_off;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const int m = warp_m0 + i * 8 + g;
      const int m1 = m1_0 + (m >> prm.tq_log2);
      const int m2 = m2_0 + (m & (tq - 1));
      if (m1 >= prm.m1_ext || m2 >= prm.m2_ext) continue;
#pragma unroll
      for (int j = 0; j < NFW; ++j) {
        const int n = n_0 + j * 8;
        if (n >= prm.n_ext) continue;
        const bool has1 = (n + 1) < prm.n_ext;
        if (prm.out_mode == 1) {
          const long long off =
              ((((long long)(m1 >> 3) * prm.nbv + (m2 >> 3)) * prm.nbv + (n >> 3)) << 9) +
              ((((m1 & 7) << 3) + (m2 & 7)) << 3) + (n & 7);
          if (has1) {
            *reinterpret_cast<double2*>(C + off) = make_double2(acc[i][j][0], acc[i][j][1]);
          } else {
            C[off] = acc[i][j][0];
          }
        } else {
          const long long base = (long long)m1 * prm.sM1 + (long long)m2 * prm.sM2;
          const long long off0 = base + (long long)(n / prm.n2_ext) * prm.sN1 + (long long)(n % prm.n2_ext) * prm.sN2;
          const long long off1 = base + (long long)((n + 1) / prm.n2_ext) * prm.sN1 +
                                 (long long)((n + 1) % prm.n2_ext) * prm.sN2;
          if (has1 && off1 == off0 + 1 && ((reinterpret_cast<uintptr_t>(C + off0) & 15) == 0)) {
            *reinterpret_cast<double2*>(C + off0) = make_double2(acc[i][j][0], acc[i][j][1]);
          } else {
            C[off0] = acc[i][j][0];
            if (has1) C[off1] = acc[i][j][1];
          }
        }
      }
    }
  }
}

template <int NF, bool kStaged, bool kTail>
__global__ void __launch_bounds__(kGemmThreads, 1)
gemm_nt_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmAT,
               const __grid_constant__ CUtensorMap tmB, const GemmParams prm) {
  constexpr int kBN = gemm_bn(NF);
  constexpr int NF0 = (NF + 1) / 2, NF1 = NF / 2;   // fragments of warp column 0 / 1
  constexpr int kStageBytes = gemm_stage_bytes(NF);
  constexpr int kStages = gemm_stages(NF, kStaged);
  static_assert(kStages >= 3, "ring too shallow");
  extern __shared__ uint8_t smem_raw[];
  // 1024-byte alignment: the 128B swizzle pattern is a function of shared address bits [4,10).
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  double* staging = reinterpret_cast<double*>(smem + kStages * kStageBytes);
  uint64_t* full_bar = reinterpret_cast<uint64_t*>(smem + kStages * kStageBytes + gemm_staging_bytes(NF, kStaged));
  uint64_t* empty_bar = full_bar + kStages;
  uint64_t* c_full = empty_bar + kStages;    // consumers -> store warp: the staging tile is complete
  uint64_t* c_empty = c_full + 1;            // store warp -> consumers: the staging tile has been read out

  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;

  if (threadIdx.x == 0) {
    for (int s = 0; s < kStages; ++s) {
      mbar_init(&full_bar[s], 1);
      mbar_init(&empty_bar[s], kConsumerWarps);
    }
    mbar_init(c_full, kConsumerWarps);
    mbar_init(c_empty, 1);
    fence_mbar_init();
  }
  if (warp == kConsumerWarps && lane == 0) {
    tma_prefetch_desc(&tmA);
    tma_prefetch_desc(&tmAT);
    tma_prefetch_desc(&tmB);
  }
  __syncthreads();

  const int tq = 1 << prm.tq_log2;
  const int tiles_per_task = prm.tiles_m1 * prm.tiles_m2 * prm.tiles_n;
  const long long total_tiles = (long long)prm.ntasks * tiles_per_task;

  if (warp >= kConsumerWarps) {
    // =========================== TMA producer (one elected lane) ===========================
    // the producer warpgroup hands its registers to the two consumer warpgroups
    asm volatile("setmaxnreg.dec.sync.aligned.u32 40;");
    if (warp == kConsumerWarps && lane == 0) {
      int stage = 0;
      uint32_t phase = 0;
      for (long long tile = blockIdx.x; tile < total_tiles; tile += gridDim.x) {
        const TileCoord tc = decode_tile(prm, tile);
        const int task_id = tc.task_id, n_t = tc.n_t, m2_t = tc.m2_t, m1_t = tc.m1_t;
        const int m1_0 = prm.m1_base + m1_t * prm.tp;
        const int m2_0 = m2_t * tq;
        const int n_0 = prm.n_base + n_t * kBN;
        const GemmTask* task = prm.tasks + task_id;
        const int nterms = task->nterms;
        for (int term = 0; term < nterms; ++term) {
          const int a_idx = task->term[term].a_idx;
          const int b_idx = task->term[term].b_idx;
          const int a_tr = task->term[term].a_transposed;
          for (int kt = 0; kt < prm.kiters; ++kt) {
            mbar_wait(&empty_bar[stage], phase ^ 1u);
            uint8_t* sA = smem + stage * kStageBytes;
            uint8_t* sB = sA + kBM * kBK * 8;
            mbar_arrive_expect_tx(&full_bar[stage], kStageBytes);
            if (!a_tr) {
              tma_load_4d(sA, &tmA, &full_bar[stage], kt * kBK, m2_0, m1_0, a_idx);
            } else {
              for (int pl = 0; pl < prm.tp; ++pl)
                tma_load_4d(sA + pl * tq * (kBK * 8), &tmAT, &full_bar[stage], kt * kBK, m1_0 + pl,
                            m2_0, a_idx);
            }
            tma_load_4d(sB, &tmB, &full_bar[stage], kt * kBK, n_0, b_idx, 0);
            if (++stage == kStages) { stage = 0; phase ^= 1u; }
          }
        }
      }
    }
    if constexpr (kStaged) {
      if (warp == kConsumerWarps + 1) {
        // =========================== store warp: staging tile -> global (bulk async copies) ===========================
        uint32_t c_phase = 0;
        constexpr int kColBlocks = kBN >> 3;
        for (long long tile = blockIdx.x; tile < total_tiles; tile += gridDim.x) {
          const TileCoord tc = decode_tile(prm, tile);
          const int task_id = tc.task_id, n_t = tc.n_t, m2_t = tc.m2_t, m1_t = tc.m1_t;
          const int m1_0 = prm.m1_out + m1_t * prm.tp;
          const int m2b_0 = (m2_t * tq) >> 3;                       // first 8-block of m2 (tq is a multiple of 8)
          const int nb_0 = (prm.n_out + n_t * kBN) >> 3;            // first 8-block of n (n_out is a multiple of 8)
          double* __restrict__ C = prm.C + prm.tasks[task_id].c_off;
          mbar_wait(c_full, c_phase);
          for (int run = lane; run < (kBM >> 3) * kColBlocks; run += 32) {
            const int rg = run / kColBlocks, cb = run - rg * kColBlocks;   // row group (8 rows), column block
            const int mrow = rg << 3;                                       // tile row of the group's first row
            const int m1 = m1_0 + (mrow >> prm.tq_log2);
            const int m2b = m2b_0 + ((mrow & (tq - 1)) >> 3);
            const int nb = nb_0 + cb;
            if (m1 >= prm.m1_ext || m2b >= prm.nbv || nb >= prm.nbv) continue;   // outside the padded F array
            const long long off = ((((long long)(m1 >> 3) * prm.nbv + m2b) * prm.nbv + nb) << 9) + ((m1 & 7) << 6);
            bulk_store_s2g(C + off, staging + ((size_t)run << 6), 512);
          }
          bulk_commit();
          bulk_wait_read_all();                  // staging has been read: the consumers may overwrite it
          __syncwarp();
          if (lane == 0) mbar_arrive(c_empty);
          c_phase ^= 1u;
        }
        bulk_wait_all();                         // the writes have completed before the CTA retires
      }
    }
    return;
  }

  // =============================== DMMA consumers (8 warps) ===============================
  asm volatile("setmaxnreg.inc.sync.aligned.u32 224;");
  // warps w and w+4 share an SM sub-partition: they take the same rows and the two column halves, so that every
  // sub-partition issues NF0 + NF1 fragments per k-step also when NF is odd.  The fragment count is a template
  // argument of the consumer loop: no predicates in the DMMA sequence.
  if constexpr (NF0 == NF1) {
    gemm_consume<NF, NF0, kStaged, kTail>(prm, smem, full_bar, empty_bar, c_full, c_empty, staging, warp, lane,
                                   (warp >> 2) * (8 * NF0), total_tiles, tiles_per_task, tq);
  } else {
    if ((warp >> 2) == 0)
      gemm_consume<NF, NF0, kStaged, kTail>(prm, smem, full_bar, empty_bar, c_full, c_empty, staging, warp, lane, 0,
                                     total_tiles, tiles_per_task, tq);
    else
      gemm_consume<NF, NF1, kStaged, kTail>(prm, smem, full_bar, empty_bar, c_full, c_empty, staging, warp, lane, 8 * NF0,
                                     total_tiles, tiles_per_task, tq);
  }
}

#endif  // __CUDACC__

// ------------------------------------------------------------------ host side
// 4-D FP64 tensor map with a (16, b1, b2, 1) box and 128-byte swizzle.
//   dims[0..3] (elements, dim 0 fastest) ; strides_bytes[1..3] (dim 0 is contiguous).
int make_tensor_map_f64(CUtensorMap* out, const void* base, const unsigned long long dims[4],
                        const unsigned long long strides_bytes[4], unsigned box1, unsigned box2);

// Launch the persistent kernel (B tile of 8*nf rows; tmB's box must have that many rows) on `stream`.
// prm.out_mode 1 (blocked F layout) selects the staged-epilogue instantiation; it needs prm.tq_log2 >= 3 and
// prm.n_out, prm.n_base multiples of 8.
// prm.tasks must stay valid until the kernel ran.
int launch_gemm_nt(int nf, const CUtensorMap& tmA, const CUtensorMap& tmAT, const CUtensorMap& tmB,
                   const GemmParams& prm, cudaStream_t stream);
// NF that minimises the modelled time (padded columns x per-tile efficiency) of an N extent.
int choose_nf(long long n_ext);
// Cover [0, n_ext) with the fewest column tiles of 8*NF, NF in [kMinNF, kMaxNF], spreading the slack evenly
// so that the padded extent is n_ext rounded up to 8 whenever n_ext >= 8*kMinNF.  At most two distinct NF
// values result; tiles of equal NF are adjacent.  Returns the number of segments written (<= 2).
struct NSegment { int n0, ntiles, nf; };
int split_n(int n_ext, NSegment seg[2], int granularity = 8);   // granularity 16: even NF only
// (tp, tq_log2) with tp * tq = 128 minimising padded rows for extents (m1_ext, m2_ext).
void choose_m_tile(int m1_ext, int m2_ext, int* tp, int* tq_log2);

// Cover the M index pairs [0, m1_ext) x [0, m2_ext) with a main range of full (tp x tq) tiles and, if m1_ext is
// not a multiple of tp, a strip of the remaining m1 rows with its own tile shape, minimising padded rows.
struct MSegment { int m1_0, tiles_m1, tp, tq_log2; };
int split_m(int m1_ext, int m2_ext, MSegment seg[2]);

int device_sm_count();

}  // namespace bqc
