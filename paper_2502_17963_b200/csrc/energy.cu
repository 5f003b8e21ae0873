// energy.cu — SURVEY.md §8(a) rows a3 + a4 (+ the reductions of a5).
//
// The W builder leaves, per triplet, three arrays in 8^3-blocked layout (each block a contiguous 4 KiB run):
//     F1 = F(i,j,k)[a,b,c],  F2 = F(i,k,j)[a,c,b],  F3 = F(j,k,i)[b,c,a],   W[a,b,c] = F1 + F2 + F3
// (see t_energy.cu).  The energy contraction needs W at all six index permutations of every point
// (Eq. (3), reading G2), so a CTA owns one *orbit* of 8^3 tiles — the up-to-six tiles
// reached from a block triple A <= B <= C by permutation — assembles the six W tiles in shared memory
// (each F tile is read exactly once from HBM), forms V on the fly from the (ov|ov) tiles and t1
// (Eqs. (6),(7); V is never stored), and reduces
//     sum_pi R_pi V_pi / D   (Eqs. (3),(4); the denominator is computed in registers, never stored).
// 35 KB of shared memory and 256 threads per CTA: several CTAs per SM, so the HBM reads of one orbit
// overlap the shared-memory and FP64 work of the others.
// Reductions are fixed-order: warp shuffle tree -> per-CTA slot -> per-triplet sum -> final sum.
#include <type_traits>

#include "kernels.cuh"

namespace bqc {

namespace {

constexpr int kET = kVB;                      // 8
constexpr int kEThreads = 256;
constexpr int kTileElems = kET * kET * kET;   // 512
// (ov|ov) / t2 operand tiles: element (u, w) of an 8 x 8 tile sits at u*8 + (w ^ u).  The two lane patterns that
// read them with 16 distinct addresses per half-warp — (u,w) = (y,z) and (z,y), z = 8 lanes, y = 2 values — then
// hit 16 distinct 8-byte bank pairs (a padded pitch of 9 left one 2-way conflict in each: 15 % of the kernel's
// shared wavefronts in the round-1 capture); the patterns through the warp-uniform x are broadcasts.
__device__ __forceinline__ int jidx(int u, int w) { return (u << 3) | (w ^ u); }
static_assert(kET == 8 && kEThreads == 256, "thread <-> element maps below assume 8^3 tiles and 256 threads");

// the six permutations of three positions; 0-2 even (identity, two cyclic), 3-5 odd (transpositions)
__device__ constexpr int kPerm[6][3] = {{0, 1, 2}, {1, 2, 0}, {2, 0, 1}, {0, 2, 1}, {2, 1, 0}, {1, 0, 2}};
// index of the ordered pair (s,t), s != t, in the (ov|ov) tile array
__device__ constexpr int kPairIdx[3][3] = {{-1, 0, 1}, {2, -1, 3}, {4, 5, -1}};

// Shared-memory position of W-tile element (X, Y, Z): linear index with its low 4 bits (the 8-byte bank
// pair) XORed by a GF(2)-linear function of (X, Y>>1).  With this mask the 16 lanes of a half-warp hit 16
// distinct bank pairs in every access pattern of the W tiles: the three assembly passes (lanes vary along
// w1,w2,v0,u0 of the F tile, written at (u,v,w), (u,w,v) and (w,u,v)) and the six permuted reads (lanes
// vary along z and y0, read at every permutation of (x,y,z)).  The columns of the mask were found by
// exhaustive search over all 2^20 linear maps.  (The claim covers the W tiles only; the operand tiles of the
// t1 / Fock terms have their own index map, jidx above.)
__device__ __forceinline__ int sw(int X, int Y, int Z) {
  const int m = ((X & 1) * 9) ^ ((X & 2) << 1) ^ ((X & 4) >> 1) ^ ((Y & 2) << 1) ^ ((Y & 4) >> 1);
  return ((X << 6) | (Y << 3) | Z) ^ m;
}

struct EnergySmem {
  double Wt[6][kTileElems];
  double Jt[3][6][kET * kET];       // [m][ordered block-position pair][jidx(local u, local w)]
  double t1s[3][3][kET];            // [which occupied (i,j,k)][block position][local]
  double epsv[3][kET];
  double red[kEThreads / 32];
};
// extra operands of the non-canonical Fock term (Eqs. (5),(7), reading G15):
// V += f[i,a] t2[j,k,b,c] + f[j,b] t2[i,k,a,c] + f[k,c] t2[i,j,a,b] — same shape as the t1 (ov|ov) term
struct FockSmem {
  double Tt[3][6][kET * kET];       // t2[y,z] tiles, indexed like Jt
  double fs[3][3][kET];             // f_ov rows, indexed like t1s
};
struct NoSmem {};

__device__ __forceinline__ size_t blk_off(int nb, int P, int Q, int R) {
  return (size_t)((P * nb + Q) * nb + R) * kTileElems;   // nb <= 1023: the block number fits 32 bits
}

}  // namespace

// Canonical kernel: 64 registers -> 4 CTAs per SM (no spills); the Fock variant keeps 80 registers / 3 CTAs.
// The shared-memory carve-out is left to the driver: forcing the maximum costs 20 % (measured), the L1 part
// serves the (ov|ov) / t1 reads.
template <bool kFock>
__global__ void __launch_bounds__(kEThreads, kFock ? 3 : 4) energy_kernel(const EnergyArgs a) {
  __shared__ EnergySmem sm;
  __shared__ typename std::conditional<kFock, FockSmem, NoSmem>::type fk;
  const int tid = threadIdx.x;
  const int orbit = blockIdx.x;
  const int tb = blockIdx.y;
  const int packed = a.orbits[orbit];
  const int blk[3] = {packed & 1023, (packed >> 10) & 1023, (packed >> 20) & 1023};
  const TripletRec tr = a.trips[tb];
  const int nb = a.nbv, v = a.v;
  const size_t fsz = (size_t)nb * nb * nb * kTileElems;
  const double* F1 = a.F + (size_t)tb * 3 * fsz;
  const double* F2 = F1 + fsz;
  const double* F3 = F2 + fsz;

  // ---- this thread's element pair of every F tile: tid bits (0..7) = (w1, w2, v0, u0, v1, v2, u1, u2)
  const int ew = (tid & 3) << 1;
  const int ev = ((tid >> 2) & 1) | (((tid >> 4) & 3) << 1);
  const int eu = ((tid >> 3) & 1) | (((tid >> 6) & 3) << 1);
  const int epair = ((eu << 6) | (ev << 3) | ew) >> 1;

  // Orbits with repeated blocks (A == B and / or B == C) reach fewer than six distinct tiles: permutation pi
  // then has the same block triple as an earlier one, canon_of(pi), and shares its W tile (neither loaded nor
  // assembled twice).  In kPerm order — (A,B,C) (B,C,A) (C,A,B) (A,C,B) (C,B,A) (B,A,C), A <= B <= C — the
  // distinct tiles are always the first nown = 6, 3 or 1 permutations.  CTA-uniform.
  const bool eAB = blk[0] == blk[1], eBC = blk[1] == blk[2], eAll = eAB && eBC;
  const int c1 = eAll ? 0 : 1, c2 = eAll ? 0 : 2, c3 = eAll ? 0 : (eAB ? 1 : (eBC ? 0 : 3)),
            c4 = eAll ? 0 : (eAB ? 2 : (eBC ? 1 : 4)), c5 = eAll ? 0 : (eAB ? 0 : (eBC ? 2 : 5));
  auto canon_of = [&](int pi) { return pi == 0 ? 0 : pi == 1 ? c1 : pi == 2 ? c2 : pi == 3 ? c3 : pi == 4 ? c4 : c5; };

  // ---- small operands (issued while the tile loads fly): t1 rows, virtual orbital energies, (ov|ov) tiles
  auto load_operands = [&]() {
    if (tid < 3 * 3 * kET) {
      const int l = tid & 7, pos = (tid >> 3) % 3, which = tid / (3 * kET);
      const int occ = which == 0 ? tr.i : (which == 1 ? tr.j : tr.k);
      const int av = blk[pos] * kET + l;
      sm.t1s[which][pos][l] = (av < v) ? a.t1[(size_t)occ * v + av] : 0.0;
      if constexpr (kFock) fk.fs[which][pos][l] = (av < v) ? a.f_ov[(size_t)occ * v + av] : 0.0;
    } else if (tid < 3 * 3 * kET + 3 * kET) {
      const int e = tid - 3 * 3 * kET;
      const int l = e & 7, pos = e >> 3;
      const int av = blk[pos] * kET + l;
      sm.epsv[pos][l] = (av < v) ? a.eps_vir[av] : 1.0;
    }
    if (a.use_t1) {
      // 18 operand tiles (3 matrices x 6 ordered block-position pairs) of 64 elements: a thread owns element
      // (lu, lw) = tid & 63 of the tiles g = (tid >> 6) + 4 it.  All loads are issued before the first store.
      const int lw = tid & 7, lu = (tid >> 3) & 7, g0 = tid >> 6;
      // (two rounds — tiles g0 + 0, 4, 8 and g0 + 12, 16 — so that the values in flight fit the register budget
      // next to the twelve F-tile loads)
      auto fill = [&](auto IT0, auto IT1) {
        constexpr int it0 = decltype(IT0)::value, it1 = decltype(IT1)::value;
        double jv[it1 - it0], tv[it1 - it0];
#pragma unroll
        for (int it = it0; it < it1; ++it) {
          const int g = g0 + 4 * it;
          jv[it - it0] = 0.0;
          tv[it - it0] = 0.0;
          if (g < 18) {
            const int m = g / 6, pr = g - 6 * m;
            // J^(0) = J_jk, J^(1) = J_ik, J^(2) = J_ij; pair index -> ordered block positions (s, t)
            const int px = (m == 0) ? tr.pj : tr.pi;
            const int py = (m == 2) ? tr.pj : tr.pk;
            const int s = pr >> 1;
            const int t = (pr & 1) ? (s == 2 ? 1 : 2) : (s == 0 ? 1 : 0);
            const int gu = blk[s] * kET + lu, gw = blk[t] * kET + lw;
            if (gu < v && gw < v) {
              jv[it - it0] = __ldg(a.J + ((size_t)(px * a.nw + py) * v + gu) * v + gw);
              if constexpr (kFock) {
                // T^(0) = t2[j,k], T^(1) = t2[i,k], T^(2) = t2[i,j]
                const int ox = (m == 0) ? tr.j : tr.i;
                const int oy = (m == 2) ? tr.j : tr.k;
                tv[it - it0] = a.dual ? -__ldg(a.t2 + (((size_t)gu * v + gw) * a.o + ox) * a.o + oy)   // -t2c[u,w,x,y]
                                      : __ldg(a.t2 + (((size_t)ox * a.o + oy) * v + gu) * v + gw);
              }
            }
          }
        }
#pragma unroll
        for (int it = it0; it < it1; ++it) {
          const int g = g0 + 4 * it;
          if (g < 18) {
            const int m = g / 6, pr = g - 6 * m;
            sm.Jt[m][pr][jidx(lu, lw)] = jv[it - it0];
            if constexpr (kFock) fk.Tt[m][pr][jidx(lu, lw)] = tv[it - it0];
          }
        }
      };
      fill(std::integral_constant<int, 0>{}, std::integral_constant<int, 3>{});
      fill(std::integral_constant<int, 3>{}, std::integral_constant<int, 5>{});
    }
  };

  // ---- load and assemble the first N W tiles: W[x,y,z] = F1[x,y,z] + F2[x,z,y] + F3[y,z,x]
  // (F tile element (eu, ev, ew): F1 -> (x,y,z), F2 -> (x,z,y), F3 -> (y,z,x)); one code copy per N so that
  // the per-tile values stay in registers
  auto assemble = [&](auto NC) {
    constexpr int N = decltype(NC)::value;
    auto load_tiles = [&](double2 (&val)[N], int phase) {
#pragma unroll
      for (int pi = 0; pi < N; ++pi) {
        const int P = blk[kPerm[pi][0]], Q = blk[kPerm[pi][1]], R = blk[kPerm[pi][2]];
        const double* src = phase == 0 ? F1 + blk_off(nb, P, Q, R)
                                       : (phase == 1 ? F2 + blk_off(nb, P, R, Q) : F3 + blk_off(nb, Q, R, P));
        val[pi] = __ldcs(reinterpret_cast<const double2*>(src) + epair);   // read once: streaming, evict-first
      }
    };
    double2 va[N], vb[N];
    load_tiles(va, 0);
    load_tiles(vb, 1);
    load_operands();
#pragma unroll
    for (int pi = 0; pi < N; ++pi) {
      sm.Wt[pi][sw(eu, ev, ew)] = va[pi].x;
      sm.Wt[pi][sw(eu, ev, ew + 1)] = va[pi].y;
    }
    load_tiles(va, 2);   // va is free again: the third class flies across the barrier
    __syncthreads();
#pragma unroll
    for (int pi = 0; pi < N; ++pi) {
      sm.Wt[pi][sw(eu, ew, ev)] += vb[pi].x;
      sm.Wt[pi][sw(eu, ew + 1, ev)] += vb[pi].y;
    }
    __syncthreads();
#pragma unroll
    for (int pi = 0; pi < N; ++pi) {
      sm.Wt[pi][sw(ew, eu, ev)] += va[pi].x;
      sm.Wt[pi][sw(ew + 1, eu, ev)] += va[pi].y;
    }
    __syncthreads();
  };
  if (eAll)
    assemble(std::integral_constant<int, 1>{});
  else if (eAB || eBC)
    assemble(std::integral_constant<int, 3>{});
  else
    assemble(std::integral_constant<int, 6>{});

  // ---- points of this thread: z = tid & 7, y = (tid >> 3) & 7, x = (tid >> 6) + 4 r
  const int lz = tid & 7, ly = (tid >> 3) & 7, lx0 = tid >> 6;
  const double dijk = a.eps_occ[tr.i] + a.eps_occ[tr.j] + a.eps_occ[tr.k];
  double acc = 0.0;
  {
    // The two points of a thread differ in one bit of x (x and x ^ 4).  Both index maps are GF(2)-linear, so
    // every shared-memory index of the second point is the first point's XOR a compile-time constant that only
    // depends on the slot x occupies after the permutation; operands that do not involve x are loaded once.
    const int l[3] = {lx0, ly, lz};
    double w0[6], w1[6];
#pragma unroll
    for (int p = 0; p < 6; ++p) {
      const int i0 = sw(l[kPerm[p][0]], l[kPerm[p][1]], l[kPerm[p][2]]);
      // flipping bit 2 of X / Y / Z moves sw() by 256^2 / 32^2 / 4 (the mask takes (X&4)>>1 and (Y&4)>>1)
      const int dx = kPerm[p][0] == 0 ? 258 : (kPerm[p][1] == 0 ? 34 : 4);
      const double* Wp = sm.Wt[canon_of(p)];
      w0[p] = Wp[i0];
      w1[p] = Wp[i0 ^ dx];
    }
    const double se0 = w0[0] + w0[1] + w0[2], so0 = w0[3] + w0[4] + w0[5];
    const double re0 = se0 - 2.0 * so0, ro0 = so0 - 2.0 * se0;
    const double se1 = w1[0] + w1[1] + w1[2], so1 = w1[3] + w1[4] + w1[5];
    const double re1 = se1 - 2.0 * so1, ro1 = so1 - 2.0 * se1;
    double s0 = 0.0, s1 = 0.0;
#pragma unroll
    for (int p = 0; p < 6; ++p) {
      // V at the permuted point: W + t1[i,a](jb|kc) + t1[j,b](ia|kc) + t1[k,c](ia|jb)   (Eqs. (6),(7))
      double v0 = w0[p], v1 = w1[p];
      if (a.use_t1) {
#pragma unroll
        for (int m = 0; m < 3; ++m) {
          const int sA = (m == 0) ? 1 : 0, sB = (m == 2) ? 1 : 2;
          const int pm = kPerm[p][m], pa = kPerm[p][sA], pb = kPerm[p][sB];
          const int ji = jidx(l[pa], l[pb]);
          const int dj = pa == 0 ? 36 : (pb == 0 ? 4 : 0);   // jidx(u ^ 4, w) = jidx ^ 36, jidx(u, w ^ 4) = jidx ^ 4
          const double* t1m = sm.t1s[m][pm];
          const double* Jm = sm.Jt[m][kPairIdx[pa][pb]];
          const double ta = t1m[l[pm]], ja = Jm[ji];
          const double tb = pm == 0 ? t1m[l[pm] + 4] : ta;
          const double jb = dj ? Jm[ji ^ dj] : ja;
          v0 = fma(ta, ja, v0);
          v1 = fma(tb, jb, v1);
          if constexpr (kFock) {
            const double* fm = fk.fs[m][pm];
            const double* Tm = fk.Tt[m][kPairIdx[pa][pb]];
            const double fa = fm[l[pm]], qa = Tm[ji];
            const double fb = pm == 0 ? fm[l[pm] + 4] : fa;
            const double qb = dj ? Tm[ji ^ dj] : qa;
            v0 = fma(fa, qa, v0);
            v1 = fma(fb, qb, v1);
          }
        }
      }
      // R at the permuted point = 3 w_p + (sum of same-parity w) - 2 (sum of opposite-parity w)   (Eq. (3))
      s0 += (3.0 * w0[p] + (p < 3 ? re0 : ro0)) * v0;
      s1 += (3.0 * w1[p] + (p < 3 ? re1 : ro1)) * v1;
    }
    // denominator (Eq. (3)) in registers
    const bool valid_yz = (blk[1] * kET + ly < v) && (blk[2] * kET + lz < v);
    const double ey = sm.epsv[1][ly], ez = sm.epsv[2][lz];
    if (valid_yz && blk[0] * kET + lx0 < v) acc += s0 / (dijk - sm.epsv[0][lx0] - ey - ez);
    if (valid_yz && blk[0] * kET + lx0 + 4 < v) acc += s1 / (dijk - sm.epsv[0][lx0 + 4] - ey - ez);
  }
  // multiplicity of the block triple under permutation (1, 2 or 6)
  const int same = (blk[0] == blk[1]) + (blk[1] == blk[2]);
  acc *= (same == 0) ? 1.0 : (same == 1 ? 0.5 : (1.0 / 6.0));

  // ---- fixed-order block reduction
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, off);
  if ((tid & 31) == 0) sm.red[tid >> 5] = acc;
  __syncthreads();
  if (tid == 0) {
    double s = 0.0;
#pragma unroll
    for (int wdx = 0; wdx < kEThreads / 32; ++wdx) s += sm.red[wdx];
    a.partial[(size_t)tb * a.norbits + orbit] = s;
  }
}

int launch_energy(const EnergyArgs& a, cudaStream_t s) {
  if (a.ntrip <= 0) return BQC_OK;
  dim3 grid(a.norbits, a.ntrip);
  if (a.use_t1 && a.f_ov)
    energy_kernel<true><<<grid, kEThreads, 0, s>>>(a);
  else
    energy_kernel<false><<<grid, kEThreads, 0, s>>>(a);
  count_launch();
  BQC_CUDA_OK(cudaGetLastError());
  return BQC_OK;
}

// ------------------------------------------------------------------ per-triplet and final sums
__global__ void reduce_triplets_kernel(const double* __restrict__ partial, const TripletRec* __restrict__ trips,
                                       int norbits, double* __restrict__ e_trip) {
  __shared__ double red[256];
  const int tb = blockIdx.x;
  const double* p = partial + (size_t)tb * norbits;
  double s = 0.0;
  for (int n = threadIdx.x; n < norbits; n += 256) s += p[n];
  red[threadIdx.x] = s;
  __syncthreads();
  for (int off = 128; off > 0; off >>= 1) {
    if (threadIdx.x < off) red[threadIdx.x] += red[threadIdx.x + off];
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    const TripletRec tr = trips[tb];
    // (2 - delta_ij - delta_jk) for i <= j <= k (reading G3)
    const double wgt = 2.0 - (tr.i == tr.j ? 1.0 : 0.0) - (tr.j == tr.k ? 1.0 : 0.0);
    e_trip[tr.index] = wgt * red[0];
  }
}

int launch_reduce_triplets(const double* partial, const TripletRec* trips, int ntrip, int norbits,
                           double* e_trip, cudaStream_t s) {
  if (ntrip <= 0) return BQC_OK;
  reduce_triplets_kernel<<<ntrip, 256, 0, s>>>(partial, trips, norbits, e_trip);
  count_launch();
  BQC_CUDA_OK(cudaGetLastError());
  return BQC_OK;
}

__global__ void final_sum_kernel(const double* __restrict__ e, long long n, double* __restrict__ out) {
  __shared__ double red[1024];
  double s = 0.0;
  for (long long i = threadIdx.x; i < n; i += 1024) s += e[i];
  red[threadIdx.x] = s;
  __syncthreads();
  for (int off = 512; off > 0; off >>= 1) {
    if (threadIdx.x < off) red[threadIdx.x] += red[threadIdx.x + off];
    __syncthreads();
  }
  if (threadIdx.x == 0) *out = red[0];
}

int launch_final_sum(const double* e_trip, long long n, double* out, cudaStream_t s) {
  final_sum_kernel<<<1, 1024, 0, s>>>(e_trip, n, out);
  count_launch();
  BQC_CUDA_OK(cudaGetLastError());
  return BQC_OK;
}

// ------------------------------------------------------------------ denominator bound on the stream (reading G10)
// out[0] = 1 if 3 max(eps_occ) - 3 min(eps_vir) >= 0 (or not comparable: NaN), else 0; out[1] = max eps_occ,
// out[2] = min eps_vir.  One block; max/min are order-independent, so the result is deterministic.
__global__ void denominator_check_kernel(const double* __restrict__ eps_occ, int o, const double* __restrict__ eps_vir,
                                         int v, double* __restrict__ out) {
  __shared__ double smax[256], smin[256];
  __shared__ int snan[256];
  double mx = -INFINITY, mn = INFINITY;
  int bad = 0;
  for (int i = threadIdx.x; i < o; i += 256) { const double e = eps_occ[i]; bad |= (e != e); mx = fmax(mx, e); }
  for (int a = threadIdx.x; a < v; a += 256) { const double e = eps_vir[a]; bad |= (e != e); mn = fmin(mn, e); }
  smax[threadIdx.x] = mx; smin[threadIdx.x] = mn; snan[threadIdx.x] = bad;
  __syncthreads();
  for (int off = 128; off > 0; off >>= 1) {
    if (threadIdx.x < off) {
      smax[threadIdx.x] = fmax(smax[threadIdx.x], smax[threadIdx.x + off]);
      smin[threadIdx.x] = fmin(smin[threadIdx.x], smin[threadIdx.x + off]);
      snan[threadIdx.x] |= snan[threadIdx.x + off];
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    const bool ok = !snan[0] && (3.0 * smax[0] - 3.0 * smin[0] < 0.0);
    out[0] = ok ? 0.0 : 1.0;
    out[1] = smax[0];
    out[2] = smin[0];
  }
}

int launch_denominator_check(const double* eps_occ, int o, const double* eps_vir, int v, double* out,
                             cudaStream_t s) {
  denominator_check_kernel<<<1, 256, 0, s>>>(eps_occ, o, eps_vir, v, out);
  count_launch();
  BQC_CUDA_OK(cudaGetLastError());
  return BQC_OK;
}

// ------------------------------------------------------------------ strictly sequential sum (cross-rank combine)
// One thread adds x[0], x[1], ... left to right: the same order (and so the same bits) as the host loop of
// bqc_sum_in_order, whatever the memory space of x.  n is a rank count, not a data size.
__global__ void ordered_sum_kernel(const double* __restrict__ x, long long n, double* __restrict__ out) {
  double s = 0.0;
  for (long long i = 0; i < n; ++i) s += x[i];
  *out = s;
}

int launch_ordered_sum(const double* x, long long n, double* out, cudaStream_t s) {
  ordered_sum_kernel<<<1, 1, 0, s>>>(x, n, out);
  count_launch();
  BQC_CUDA_OK(cudaGetLastError());
  return BQC_OK;
}

// ------------------------------------------------------------------ dense W / V of one triplet (debug)
__global__ void assemble_wv_kernel(const double* __restrict__ F, int nb, int v, const double* __restrict__ Jjk,
                                   const double* __restrict__ Jik, const double* __restrict__ Jij,
                                   const double* __restrict__ t1i, const double* __restrict__ t1j,
                                   const double* __restrict__ t1k, const double* __restrict__ Tjk,
                                   const double* __restrict__ Tik, const double* __restrict__ Tij,
                                   const double* __restrict__ fi, const double* __restrict__ fj,
                                   const double* __restrict__ fk, double* __restrict__ W,
                                   double* __restrict__ V) {
  const size_t fsz = (size_t)nb * nb * nb * kTileElems;
  const long long total = (long long)v * v * v;
  for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < total;
       e += (long long)gridDim.x * blockDim.x) {
    const int c = (int)(e % v);
    const int b = (int)((e / v) % v);
    const int a = (int)(e / ((long long)v * v));
    auto at = [&](const double* Fx, int p, int q, int r) {
      return Fx[blk_off(nb, p >> 3, q >> 3, r >> 3) + ((((p & 7) << 3) | (q & 7)) << 3 | (r & 7))];
    };
    const double w = at(F, a, b, c) + at(F + fsz, a, c, b) + at(F + 2 * fsz, b, c, a);
    if (W) W[e] = w;
    if (V) {
      double val = w + t1i[a] * Jjk[(size_t)b * v + c] + t1j[b] * Jik[(size_t)a * v + c] +
                   t1k[c] * Jij[(size_t)a * v + b];
      if (fi) val += fi[a] * Tjk[(size_t)b * v + c] + fj[b] * Tik[(size_t)a * v + c] + fk[c] * Tij[(size_t)a * v + b];
      V[e] = val;
    }
  }
}

int launch_assemble_wv(const double* F, int nbv, int v, const double* J, int nw, int pi, int pj, int pk,
                       const double* t1i, const double* t1j, const double* t1k, const double* t2, int o, int i,
                       int j, int k, const double* f_ov, double* W, double* V, cudaStream_t s) {
  const size_t v2 = (size_t)v * v;
  const bool fock = f_ov != nullptr;
  assemble_wv_kernel<<<1024, 256, 0, s>>>(F, nbv, v, J + ((size_t)pj * nw + pk) * v2,
                                          J + ((size_t)pi * nw + pk) * v2, J + ((size_t)pi * nw + pj) * v2,
                                          t1i, t1j, t1k, fock ? t2 + ((size_t)j * o + k) * v2 : nullptr,
                                          fock ? t2 + ((size_t)i * o + k) * v2 : nullptr,
                                          fock ? t2 + ((size_t)i * o + j) * v2 : nullptr,
                                          fock ? f_ov + (size_t)i * v : nullptr, fock ? f_ov + (size_t)j * v : nullptr,
                                          fock ? f_ov + (size_t)k * v : nullptr, W, V);
  count_launch();
  BQC_CUDA_OK(cudaGetLastError());
  return BQC_OK;
}

}  // namespace bqc
