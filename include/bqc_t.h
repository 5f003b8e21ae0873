/*
 * bqc_t.h — C ABI of the B200-native closed-shell RHF (T) energy library (libbqc_t.so).
 *
 * What is computed (citations: /root/reference/PAPER.md = ByteQC, arxiv 2502.17963, §2.4.2,
 * lines 282-305, Eqs. (2)-(7); readings G1-G14 in DESIGN.md / SURVEY.md §8(c)):
 *
 *   integrals   (pq|rs) = sum_Q B[Q,p,q] B[Q,r,s]                      (exact DF)
 *   W_ijk[abc]  = P sum_d (ia|bd) t2[k,j,c,d] - P sum_l (ia|jl) t2[l,k,b,c]          Eq. (2)
 *                 (P = the 6 simultaneous permutations of (i,a),(j,b),(k,c))
 *   V_ijk[abc]  = W + t1[i,a](jb|kc) + t1[j,b](ia|kc) + t1[k,c](ia|jb)              Eqs. (6),(7)
 *                 [+ f[i,a] t2[j,k,b,c] + f[j,b] t2[i,k,a,c] + f[k,c] t2[i,j,a,b]    Eqs. (5),(7), only when
 *                    bqc_t_opts.f_ov is given: non-canonical reference, SURVEY.md §8(f) NEXT-3]
 *   R_ijk[abc]  = 4W[abc] + W[bca] + W[cab] - 2(W[acb] + W[cba] + W[bac])           Eq. (3)
 *   D_ijk[abc]  = eps_i + eps_j + eps_k - eps_a - eps_b - eps_c                      Eq. (3)
 *   e_ijk       = (2 - d_ij - d_jk) sum_abc R V / D            (i <= j <= k)        Eq. (4)
 *   E(T)        = sum_{i<=j<=k} e_ijk
 *
 * Conventions common to every entry point
 *   - All arrays are FP64, C-contiguous (last index fastest), 8-byte aligned.
 *   - "device" pointers are CUDA device memory on the current device and stay owned by the
 *     caller; the library only reads them and they must stay valid until the call returns.
 *   - `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).  All work is
 *     ordered after prior work on `stream`; calls return after the results reached the host
 *     (they synchronise `stream` and the library's internal helper stream only).
 *   - No exceptions cross the ABI, there is NO CPU fallback: on any error the call returns the
 *     error code (or NaN for the double-returning form) and bqc_last_error() reports it.
 *   - Preconditions (not checked): t2[i,j,a,b] == t2[j,i,b,a]; B_oo, B_vv symmetric in their last
 *     two indices.  If violated the result is unspecified (reading G14).
 *   - Determinism: identical inputs and options give a bit-identical result on the same
 *     build/GPU (fixed-order reductions, no floating-point atomics).
 */
#ifndef BQC_T_H
#define BQC_T_H

#include <stddef.h>

#if defined(__GNUC__)
#define BQC_API __attribute__((visibility("default")))
#else
#define BQC_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

/* Error codes (bqc_last_error / return values). */
enum {
  BQC_OK = 0,
  BQC_ERR_INVALID_SIZE = 1,    /* nocc, nvir or naux <= 0, or option out of range          */
  BQC_ERR_NULL_POINTER = 2,    /* a required pointer is NULL                                */
  BQC_ERR_NOT_DEVICE_PTR = 3,  /* an array pointer is not device memory (or not host, for _host) */
  BQC_ERR_MISALIGNED = 4,      /* an array pointer is not 8-byte aligned                    */
  BQC_ERR_WORKSPACE = 5,       /* caller workspace too small / allocation failed            */
  BQC_ERR_CUDA = 6,            /* a CUDA runtime/driver call failed (see bqc_error_detail)  */
  BQC_ERR_DEVICE = 7,          /* current device is not sm_100 (B200)                       */
  BQC_ERR_DENOMINATOR = 8,     /* 3*max(eps_occ) - 3*min(eps_vir) >= 0: D may vanish (G10)  */
  BQC_ERR_INVALID_OPTION = 9   /* bqc_t_opts field out of range                             */
};

/* Options of bqc_t_energy_ex.  Zero-initialise for defaults. */
typedef struct bqc_t_opts {
  int occ_block;     /* occupied block size Bo of the slab cache (0 = auto from workspace_gib).  4*Bo
                        (vv|ov) slabs and the B~ / (ov|ov) blocks of 16 Bo^2 orbital pairs are resident
                        at a time; the full O(o v^3) and O(o^2 v^2) tensors never are.          */
  int occ_lo;        /* restrict to triplets with occ_lo <= i <= j <= k < occ_hi;            */
  int occ_hi;        /*   occ_lo = occ_hi = 0 means all occupied orbitals.                   */
  int shard_rank;    /* multi-GPU sharding: this call evaluates the triplets whose index     */
  int shard_count;   /*   (bqc_t_triplet_index) % shard_count == shard_rank.  0 -> 1.
                        (BQC_T_FLAG_SHARD_BLOCKS deals whole block triples instead.)         */
  int max_batch;     /* triplets per W-builder launch (0 = auto from memory)                 */
  int flags;         /* BQC_T_FLAG_* below                                                   */
  int workspace_gib; /* soft cap, in GiB, on the buffers whose size follows occ_block (slab cache + pair
                        blocks) when occ_block = 0; 0 = 36.  The fixed part (K-major DF copies, one batch
                        of F arrays) comes on top: bqc_t_workspace_bytes reports the total.          */
  const double* f_ov;/* non-canonical reference (Eqs. (5),(7); reading G15): the
                        occupied-virtual Fock block f[i,a], [nocc][nvir], caller-owned, read-only;
                        DEVICE memory for bqc_t_energy_ex, HOST memory for bqc_t_energy_host.
                        V gains f[i,a] t2[j,k,b,c] + f[j,b] t2[i,k,a,c] + f[k,c] t2[i,j,a,b].
                        NULL (default) = canonical RHF, F_ov = 0 (reading G7).               */
} bqc_t_opts;

enum {
  BQC_T_FLAG_NO_T1 = 1,         /* drop the t1 (E[5]) and Fock terms: V = W (E[4]-only checks) */
  BQC_T_FLAG_PROFILE = 2,       /* bracket every kernel group with CUDA events on its launching
                                   stream; read the sums with bqc_t_last_profile             */
  BQC_T_FLAG_ABC_DRIVEN = 4,    /* abc-driven schedule (the paper's loop order; SURVEY.md
                                   §8(f) NEXT-2): the outer loop runs over virtual triples a<=b<=c with all
                                   o^3 occupied triples inside, instead of occupied triplets i<=j<=k with
                                   all v^3 virtual triples inside.  Same E(T) up to summation order; the
                                   resident pieces are o^2 (v+o) per virtual orbital of a block instead of
                                   v^2 (v+o) per occupied orbital, and O(Bv^2 o (v+o)) for the pairs of the
                                   4 resident virtual blocks of Bv orbitals — nothing of size o v^3 or
                                   v^2 o^2 is stored, no transposed copy of t2 or B_vv is made — which is
                                   what large virtual spaces (cc-pVTZ/QZ-shaped inputs) need.  With this flag
                                   occ_block / occ_lo / occ_hi / shard_* refer to the VIRTUAL index,
                                   e_triplet_dev has bqc_t_num_triplets(nvir) entries indexed by
                                   bqc_t_triplet_index(nvir, a, b, c) and holds the weighted
                                   per-virtual-triple contributions (2 - d_ab - d_bc) sum_ijk R V / D, and
                                   bqc_t_flops counts 12 o^3 (v+o) per virtual triple.                   */
  BQC_T_FLAG_SHARD_BLOCKS = 8   /* multi-GPU sharding by whole block triples instead of single triplets: with
                                   shard_count > 1 the block triples (I <= J <= K blocks of occ_block orbitals)
                                   are dealt to the ranks largest first, each to the least-loaded rank (a
                                   deterministic function of window, occ_block and shard_count that every rank
                                   computes identically), and a rank forms only the (vv|ov) slabs its own block
                                   triples need — the per-triplet modulo makes every shard form every slab.
                                   Shards are disjoint and cover every triplet once; per-triplet values are the
                                   same bits.  With occ_block = 0 the block size is lowered from the
                                   memory-derived one until the deal is within 3 % of even.
                                   bqc_t_triplet_owner_ex describes the split, bqc_t_flops each rank's share. */
};

/* ---- host-only helpers (no GPU needed) -------------------------------------------------- */

/* o(o+1)(o+2)/6 = number of i<=j<=k triplets. */
BQC_API size_t bqc_t_num_triplets(int nocc);
/* Lexicographic index of (i,j,k), 0 <= i <= j <= k < nocc; (size_t)-1 if out of range. */
BQC_API size_t bqc_t_triplet_index(int nocc, int i, int j, int k);
/* Rank that evaluates triplet (i,j,k) under `shard_count`-way sharding (-1 on bad args). */
BQC_API int bqc_t_triplet_owner(int nocc, int shard_count, int i, int j, int k);
/* Rank that evaluates triplet (i,j,k) under the sharding `opts` describes: the per-triplet modulo above, or,
   with BQC_T_FLAG_SHARD_BLOCKS, the owner of its block triple (window, occ_block and shard_count taken from
   opts; shard_rank ignored).  With BQC_T_FLAG_ABC_DRIVEN (i,j,k) is a virtual triple a<=b<=c.  -1 if the
   triplet is outside the window or an argument is invalid.  This is the host description of the split the
   multi-GPU path uses. */
BQC_API int bqc_t_triplet_owner_ex(int nocc, int nvir, int naux, const bqc_t_opts* opts, int i, int j, int k);
/* Algorithmic FP64 flop count of the W builder over the selected triplets:
   [#triplets(i<=j<=k, not i=j=k) in window/shard] * 12 v^3 (v+o). */
BQC_API double bqc_t_flops(int nocc, int nvir, const bqc_t_opts* opts);
/* Occupied block size the scheduler will use (resolves opts->occ_block == 0). */
BQC_API int bqc_t_plan_occ_block(int nocc, int nvir, int naux, const bqc_t_opts* opts);
/* Bytes of device workspace bqc_t_energy_ex needs for these sizes/options. */
BQC_API size_t bqc_t_workspace_bytes(int nocc, int nvir, int naux, const bqc_t_opts* opts);

/* The fixed-order sum that closes the multi-GPU path (the
   independent pieces of (T) are split over GPUs and only their partial energies are combined):
   *out_host = x[0] + x[1] + ... + x[n-1], added strictly left to right in FP64.  x may be a HOST or a
   DEVICE pointer (detected; a device array is summed by a one-thread kernel on `stream`, in the same
   order, so both give the same bits).  Used on the rank-ordered all-gather of the per-rank partial
   energies, so that every rank returns an identical E(T).  Usable without a GPU for host arrays. */
BQC_API int bqc_sum_in_order(const double* x, size_t n, double* out_host, void* stream);

/* The one entry point that allocates nothing (for callers that cannot call cudaMalloc: code under CUDA-graph
   capture, tight serving loops, harnesses that forbid it).  A two-stage variant of the path's fixed-order final
   sum: *out_dev = sum of x_dev[0 .. n), both DEVICE pointers on the current device,
   enqueued on `stream` without any host synchronisation (the result is ready when the stream reaches that
   point).  One CTA per 4096-element chunk writes its partial sum into a file-scope `static __device__` scratch
   array of 4096 doubles (32 KiB, held by every GPU that loads the library until the process exits), one CTA adds
   the partials; the order of additions depends on n only, so equal inputs give equal bits.  The call performs
   no cudaMalloc / cudaFree / cudaMallocAsync and calls no allocating library routine.
   Limit: n <= bqc_sum_fixed_noalloc_max() = 16 777 216 elements; larger n returns BQC_ERR_INVALID_SIZE.
   All calls on a device share the scratch array (it keeps the last call's contents; nothing in it has to start
   at zero: every slot a call reads it has written itself).  Calls that overlap on the GPU — different streams,
   or several host threads on one device — race on it: order them on one stream or with events. */
BQC_API int bqc_sum_fixed_noalloc(const double* x_dev, size_t n, double* out_dev, void* stream);
BQC_API size_t bqc_sum_fixed_noalloc_max(void);

BQC_API int bqc_last_error(void);                 /* thread-local code of the last failing call (0 = none) */
BQC_API const char* bqc_error_string(int code);   /* static description of an error code */
BQC_API const char* bqc_error_detail(void);       /* thread-local detail text of the last error ("" if none) */
BQC_API const char* bqc_version(void);

/* ---- the (T) energy ------------------------------------------------------------------------ */

/* E(T) in Hartree; NaN on error.  All array arguments are DEVICE pointers:
     eps_occ [nocc], eps_vir [nvir], t1 [nocc][nvir], t2 [nocc][nocc][nvir][nvir],
     B_oo [naux][nocc][nocc], B_ov [naux][nocc][nvir]  (B_ov[Q,i,a] = B[Q,i,nocc+a]),
     B_vv [naux][nvir][nvir].
   Workspace is allocated on the device internally; it is freed before return when larger than 2 GiB and
   otherwise kept with the thread's cached plan for the next call (bqc_release_cached frees it).
   nocc == 1 is valid and returns exactly 0.0 (no triples with two electrons). */
BQC_API double bqc_t_energy(int nocc, int nvir, int naux,
                    const double* eps_occ, const double* eps_vir,
                    const double* t1, const double* t2,
                    const double* B_oo, const double* B_ov, const double* B_vv,
                    void* stream);

/* Same computation with options, caller workspace and per-triplet output.
     workspace       device, >= bqc_t_workspace_bytes(...) bytes, 256-byte aligned; NULL = allocate
                     internally (workspace_bytes ignored).
     e_total_host    HOST pointer, receives the sum of the selected e_ijk (this shard/window).
     e_triplet_dev   DEVICE pointer [bqc_t_num_triplets(nocc)] or NULL; receives e_ijk at
                     bqc_t_triplet_index(i,j,k); entries not selected by the window/shard and
                     the diagonal i=j=k entries are written as 0.
   Returns BQC_OK or an error code. */
BQC_API int bqc_t_energy_ex(int nocc, int nvir, int naux,
                    const double* eps_occ, const double* eps_vir,
                    const double* t1, const double* t2,
                    const double* B_oo, const double* B_ov, const double* B_vv,
                    const bqc_t_opts* opts, void* workspace, size_t workspace_bytes,
                    double* e_total_host, double* e_triplet_dev, void* stream);

/* Reusable plan (PAPER.md:177 on the cost of allocations inside a loop): everything of an
   evaluation that does not depend on the VALUES of the inputs — workspace (caller's, or allocated once here
   when workspace == NULL), helper stream, events, tensor maps, the block-triple schedule — is built once by
   bqc_t_plan_create and reused by every bqc_t_plan_execute on the same device.  Array arguments and results
   are as for bqc_t_energy_ex; f_ov must be non-NULL exactly when the plan was created with opts->f_ov set
   (only its NULL-ness is recorded at creation).  A plan is used by one thread at a time.
   bqc_t_energy_ex keeps the plan of the thread's last call and reuses it when sizes, options, workspace and
   device repeat (a plan that owns more than 2 GiB of workspace is dropped when its call returns);
   bqc_release_cached() frees it. */
typedef struct bqc_t_plan_s* bqc_t_plan;
/* Short schedules (at most 8 W-builder launches and 2 block triples, BQC_T_FLAG_PROFILE not set) are captured
   into a CUDA graph on an internal stream the first time a plan sees a set of argument pointers and replayed
   on the caller's stream afterwards; the replay reads the current VALUES behind those pointers, a different
   pointer re-captures.  Results are the same bits as the eager path.  Every call still ends with one host
   synchronisation of `stream` (the result travels to the host), so these entry points cannot themselves run
   inside a caller's stream capture. */
BQC_API int bqc_t_plan_create(int nocc, int nvir, int naux, const bqc_t_opts* opts,
                      void* workspace, size_t workspace_bytes, bqc_t_plan* plan_out);
BQC_API int bqc_t_plan_execute(bqc_t_plan plan,
                      const double* eps_occ, const double* eps_vir, const double* t1, const double* t2,
                      const double* B_oo, const double* B_ov, const double* B_vv, const double* f_ov,
                      double* e_total_host, double* e_triplet_dev, void* stream);
BQC_API void bqc_t_plan_destroy(bqc_t_plan plan);
BQC_API size_t bqc_t_plan_workspace_bytes(bqc_t_plan plan);   /* bytes of device workspace the plan uses */
BQC_API void bqc_release_cached(void);                         /* drop this thread's cached plan */

/* Timing of the last bqc_t_energy_ex call of this thread that had BQC_T_FLAG_PROFILE set, measured
   with CUDA events on the streams the kernels were launched on.  Fills up to n (<= 9) doubles:
     [0] W-builder (tile-GEMM) kernel milliseconds, summed over launches   [1] number of those launches
     [2] energy-contraction + per-triplet reduction kernel milliseconds     [3] number of those launches
     [4] slab-former + B~/J pair-block former milliseconds (DF GEMMs)       [5] number of slab blocks formed
     [6] input repacking milliseconds                                       [7] whole call, first to last kernel
     [8] number of library kernels launched by the call (counted whether or not PROFILE was set)
   Returns the number of values written (n <= 9). */
BQC_API int bqc_t_last_profile(double* out, int n);

/* End-to-end form: every array argument is a HOST pointer (pinned or pageable).  Inputs are
   copied to the device, E(T) is evaluated by the same kernels, the scalar (and, if
   e_triplet_host != NULL, the [num_triplets] per-triplet array) is copied back.
   With an occupied window (opts->occ_lo/occ_hi, ijk-driven schedule) only the rows t2[x,:,:,:],
   occ_lo <= x < occ_hi, are copied: a window reads no other part of t2.
   h2d_bytes / d2h_bytes (may be NULL) receive the bytes actually moved each way. */
BQC_API int bqc_t_energy_host(int nocc, int nvir, int naux,
                      const double* eps_occ, const double* eps_vir,
                      const double* t1, const double* t2,
                      const double* B_oo, const double* B_ov, const double* B_vv,
                      const bqc_t_opts* opts, double* e_total_host, double* e_triplet_host,
                      size_t* h2d_bytes, size_t* d2h_bytes, void* stream);

/* ---- intermediates of single steps, for parity tests ---------- */

/* Row a1: the DF slabs of occupied x (and pair x,y).  Any output pointer may be NULL.
     I_dev [nvir][nvir][nvir]   I_x[u,b,d]  = (x u|b d)
     O_dev [nocc][nvir]         O_xy[l,u]   = (x u|y l)
     J_dev [nvir][nvir]         J_xy[u,w]   = (x u|y w)
   computed by the same slab-former kernels as the energy path. */
BQC_API int bqc_t_debug_slabs(int nocc, int nvir, int naux,
                      const double* t2, const double* B_oo, const double* B_ov, const double* B_vv,
                      int x, int y, double* I_dev, double* O_dev, double* J_dev, void* stream);

/* Rows a2+a3: W_ijk and V_ijk of one triplet, dense [nvir][nvir][nvir] device outputs (either
   may be NULL), produced by the same slab former, W builder and V assembly as the energy path.
   (i, j, k) need not be ordered.  f_ov: DEVICE [nocc][nvir] occupied-virtual Fock block or NULL
   (see bqc_t_opts.f_ov); it enters V only. */
BQC_API int bqc_t_debug_wv(int nocc, int nvir, int naux,
                   const double* eps_occ, const double* eps_vir,
                   const double* t1, const double* t2,
                   const double* B_oo, const double* B_ov, const double* B_vv,
                   const double* f_ov, int i, int j, int k, double* W_dev, double* V_dev, void* stream);

/* ---- closed-shell DF-MP2 energy ------------------------------------ */

/* PAPER.md:252-258 (§2.3, Eq. (1)), unrestricted closed-shell sum (reading M1 in DESIGN.md):
     J_ij[a,b] = (ia|jb) = sum_Q B_ov[Q,i,a] B_ov[Q,j,b]                       (exact DF)
     e_ij      = sum_ab J_ij[a,b] (2 J_ij[a,b] - J_ij[b,a]) / (eps_i + eps_j - eps_a - eps_b)
     E_MP2     = sum_{i,j} e_ij = sum_{i<=j} (2 - d_ij) e_ij                   (e_ij = e_ji)
   The (ov|ov) integrals are formed block by block with the library's TMA + DMMA tile GEMM and never
   stored whole; the denominator is evaluated in registers from the orbital energies.
   Options, zero-initialise for defaults. */
typedef struct bqc_mp2_opts {
  int occ_block;     /* occupied orbitals i per (ov|ov) block (0 = auto: block buffer <= 2 GiB)     */
  int shard_rank;    /* multi-GPU sharding: this call evaluates the occupied blocks whose number     */
  int shard_count;   /*   % shard_count == shard_rank (all pairs i <= j of those rows i).  0 -> 1.  */
  int flags;         /* BQC_T_FLAG_PROFILE: time the kernel groups, read with bqc_mp2_last_profile  */
  void* workspace;   /* optional caller-owned DEVICE scratch, 256-byte aligned, >= bqc_mp2_workspace_bytes; */
  size_t workspace_bytes; /* NULL / 0: one block is allocated internally and freed before return      */
} bqc_mp2_opts;

/* E_MP2 in Hartree; NaN on error.  DEVICE pointers: eps_occ [nocc], eps_vir [nvir],
   B_ov [naux][nocc][nvir].  Device scratch is allocated internally and freed before return.
   Error behaviour as bqc_t_energy; BQC_ERR_DENOMINATOR if 2*max(eps_occ) - 2*min(eps_vir) >= 0. */
BQC_API double bqc_mp2_energy(int nocc, int nvir, int naux, const double* eps_occ, const double* eps_vir,
                      const double* B_ov, void* stream);

/* Same with options and per-pair output.
     e_total_host  HOST pointer; receives sum_{i<=j, i in this shard's blocks} (2 - d_ij) e_ij.
     e_pair_dev    DEVICE pointer [nocc][nocc] or NULL; receives the unweighted e_ij at [i][j] AND [j][i]
                   for every pair this call evaluated, 0 elsewhere.
   Returns BQC_OK or an error code. */
BQC_API int bqc_mp2_energy_ex(int nocc, int nvir, int naux, const double* eps_occ, const double* eps_vir,
                      const double* B_ov, const bqc_mp2_opts* opts, double* e_total_host,
                      double* e_pair_dev, void* stream);

/* End-to-end form: HOST pointers in, H2D of the three inputs and D2H of the scalar (and of the
   [nocc][nocc] pair matrix when e_pair_host != NULL) inside the call. */
BQC_API int bqc_mp2_energy_host(int nocc, int nvir, int naux, const double* eps_occ, const double* eps_vir,
                        const double* B_ov, const bqc_mp2_opts* opts, double* e_total_host,
                        double* e_pair_host, size_t* h2d_bytes, size_t* d2h_bytes, void* stream);

/* Algorithmic FP64 flop count of the (ov|ov) contraction over the pairs i <= j:
   o(o+1)/2 * 2 v^2 X (the energy reduction, ~8 flops per element, is not counted). */
BQC_API double bqc_mp2_flops(int nocc, int nvir, int naux);
/* Bytes of device scratch bqc_mp2_energy_ex needs for these sizes/options (0 on bad arguments). */
BQC_API size_t bqc_mp2_workspace_bytes(int nocc, int nvir, int naux, const bqc_mp2_opts* opts);
/* Occupied block size bqc_mp2_energy_ex will use (resolves opts->occ_block == 0); -1 on bad sizes. */
BQC_API int bqc_mp2_plan_occ_block(int nocc, int nvir, int naux, const bqc_mp2_opts* opts);
/* Timing of this thread's last profiled bqc_mp2_energy_ex call (CUDA events on the launch stream):
     [0] (ov|ov) tile-GEMM ms  [1] its launches  [2] pair-energy + reduction kernel ms  [3] their launches
     [4] whole call ms         [5] library kernels launched.   Returns the number of values written. */
BQC_API int bqc_mp2_last_profile(double* out, int n);

/* ---- building blocks exposed for measurement ------------------------------------------------ */

/* Host-only: the tiling the W-builder GEMM uses for nvir virtual orbitals (DESIGN.md §2.3 "exact tiling").
   out[0..5]  = up to two column segments  (n0, ntiles, NF): columns [n0, n0 + ntiles*8*NF)
   out[6..13] = up to two row segments     (m1_0, tiles_m1, tp, tq): rows m1 in [m1_0, m1_0 + tiles_m1*tp),
                each tile tp (m1) x tq (m2), tp*tq = 128
   Returns 10*(number of column segments) + (number of row segments), or -1 on bad arguments (n >= 14). */
BQC_API int bqc_debug_tiling(int nvir, int* out, int n);

/* C[M][N] (ldc) = A[M][K] (lda) * B[N][K]^T (ldb), FP64, device pointers, the library's TMA +
   DMMA tile kernel.  lda, ldb must be multiples of 2 (16-byte rows), K is zero-padded
   internally to a multiple of 16 by TMA out-of-bounds fill.  Returns BQC_OK or an error. */
BQC_API int bqc_dgemm_nt(int M, int N, int K, const double* A, int lda, const double* B, int ldb,
                 double* C, int ldc, void* stream);

/* Register-resident FP64 peak microbenchmarks on all SMs: run for about
   `seconds` and return the sustained TFLOP/s.  kind: 0 = DMMA (mma.sync m8n8k4 f64),
   1 = DFMA (fma.rn.f64), 2 = both pipes in the same warps.  Negative on error. */
BQC_API double bqc_fp64_peak_tflops(int kind, double seconds, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* BQC_T_H */
