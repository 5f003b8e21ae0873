// kernels.cuh — launchers of the non-GEMM kernels (repacking, energy contraction, reductions).
#pragma once
#include "common.cuh"

namespace bqc {

// out[row(r)][q] (pitch qp, zero for nq <= q < qp) = in[q][r0 + r], r < nr   (in: [nq][in_pitch] row-major).
// row(r) = r, or with perm_v > 0 the pair-transposed row of column c = r0 + r = i*perm_v + a: a*perm_o + i.
int launch_transpose_pad(const double* in, long long in_pitch, long long r0, long long nr, double* out, int nq,
                         int qp, int perm_v, int perm_o, cudaStream_t s);

// out[b][c][r] = scale * in[b][r][c]   (in: [batch][nr][nc] row-major; nr <= 32*65535, batch <= 65535)
int launch_transpose_scale(const double* in, double* out, int batch, long long nr, long long nc, double scale,
                           cudaStream_t s);

// Particle columns of the B~ pair block (z0..z0+nz) x (y0..y0+ny) at slots (sz0.., sy0..):
//   B~[(sz0+z)*nslots + sy0+y][r][d] = t2'[z0+z][y0+y][r][d], d < v (row pitch kp; columns >= v untouched),
// t2' = the caller's t2 (dual = false) or its particle-hole dual -t2[r][d][z][y] (dual = true; o, v are the
// pipeline-space extents, the caller's array is [v][v][o][o]).
int launch_btilde_t2(const double* t2, double* btil, int o, int v, int kp, int nslots, int z0, int nz, int y0,
                     int ny, int sz0, int sy0, bool dual, cudaStream_t s);

// slab[slot0 + s][p][q][v + l] = -t2'[x0 + s][l][p][q]  for s < nx, l < o   (row pitch kp).
int launch_slab_holes(const double* t2, double* slabs, int o, int v, int kp, int x0, int nx, int slot0, bool dual,
                      cudaStream_t s);

// Edge of the cubic virtual-index blocks of the F layout (GEMM epilogue writes, energy kernel reads).
constexpr int kVB = 8;

// One entry per triplet of a batch.
struct TripletRec {
  int i, j, k;        // outer-index orbitals, i <= j <= k
  int pi, pj, pk;     // slab-cache slots of i, j, k (B~ / J pair blocks are indexed by slot pairs)
  long long index;    // bqc_t_triplet_index(i, j, k)
};

struct EnergyArgs {
  const double* F;          // [ntrip][3][nbv^3][8^3] blocked F(i,j,k), F(i,k,j), F(j,k,i)
  const TripletRec* trips;  // [ntrip]
  const int* orbits;        // [norbits] packed A | B<<10 | C<<20, A <= B <= C
  const double* J;          // [nw*nw][v][v]   J_xy[u,w] = (xu|yw), indexed by the slot pair (nw = nslots)
  const double* t1;         // [o][v]
  const double* eps_occ;    // [o]
  const double* eps_vir;    // [v]
  const double* t2;         // [o][o][v][v]   (Fock term only)
  const double* f_ov;       // [o][v] occupied-virtual Fock block, or NULL (canonical reference)
  double* partial;          // [ntrip][norbits]
  int ntrip, norbits, nbv, v, nw, use_t1, o;
  int dual;                 // abc-driven: t2 is the caller's [v][v][o][o] array, t2'[x,y,u,w] = -t2[u,w,x,y]
};
int launch_energy(const EnergyArgs& a, cudaStream_t s);

// e_trip[trips[t].index] = weight(i,j,k) * sum_orbits partial[t][:]   (fixed order)
int launch_reduce_triplets(const double* partial, const TripletRec* trips, int ntrip, int norbits,
                           double* e_trip, cudaStream_t s);
// *out = sum_n e_trip[n] in a fixed order (single block)
int launch_final_sum(const double* e_trip, long long n, double* out, cudaStream_t s);

// out[0] = 1 if 3 max(eps_occ) - 3 min(eps_vir) >= 0 or a NaN is present (denominators may vanish), else 0;
// out[1] = max eps_occ, out[2] = min eps_vir   (device pointers, evaluated on the stream)
int launch_denominator_check(const double* eps_occ, int o, const double* eps_vir, int v, double* out,
                             cudaStream_t s);

// *out = x[0] + x[1] + ... + x[n-1], one thread, left to right (device pointers)
int launch_ordered_sum(const double* x, long long n, double* out, cudaStream_t s);

// dense W / V [v][v][v] of one triplet from its three blocked F arrays (debug / parity of rows a2, a3)
int launch_assemble_wv(const double* F, int nbv, int v, const double* J, int nw, int pi, int pj, int pk,
                       const double* t1i, const double* t1j, const double* t1k, const double* t2, int o, int i,
                       int j, int k, const double* f_ov, double* W, double* V, cudaStream_t s);

// strided 3-D copy out[a][b][c] = in[a*sa + b*sb + c*sc], used to unpad debug slabs
int launch_copy3(const double* in, long long sa, long long sb, long long sc, double* out, int na, int nb,
                 int nc, cudaStream_t s);

double run_fp64_peak(int kind, double seconds, cudaStream_t s);

}  // namespace bqc
