// kernels.cuh — launchers of the non-GEMM kernels (repacking, energy contraction, reductions).
#pragma once
#include "common.cuh"

namespace bqc {

// out[r][q] (pitch qp, zero for q >= nq) = in[q][r]        (in: [nq][nr] row-major)
int launch_transpose_pad(const double* in, double* out, int nq, int nr, int qp, cudaStream_t s);

// out[b][c][r] = scale * in[b][r][c]   (in: [batch][nr][nc] row-major; nr <= 32*65535, batch <= 65535)
int launch_transpose_scale(const double* in, double* out, int batch, long long nr, long long nc, double scale,
                           cudaStream_t s);

// Btil[pz*na + py][r][d] = t2[act[pz]][act[py]][r][d], d < v  (row pitch kp).  Columns >= v untouched.
int launch_btilde_t2(const double* t2, double* btil, int o, int v, const int* act_dev, int na, int kp,
                     cudaStream_t s);

// slab[slot0 + s][p][q][v + l] = -t2[x0 + s][l][p][q]  for s < nx, l < o   (row pitch kp).
int launch_slab_holes(const double* t2, double* slabs, int o, int v, int kp, int x0, int nx,
                      int slot0, cudaStream_t s);

// Edge of the cubic virtual-index blocks of the F layout (GEMM epilogue writes, energy kernel reads).
constexpr int kVB = 8;

// One entry per triplet of a batch.
struct TripletRec {
  int i, j, k;        // occupied indices, i <= j <= k
  int pi, pj, pk;     // indices relative to the occupied window (i - lo, ...)
  long long index;    // bqc_t_triplet_index(i, j, k)
};

struct EnergyArgs {
  const double* F;          // [ntrip][3][nbv^3][8^3] blocked F(i,j,k), F(i,k,j), F(j,k,i)
  const TripletRec* trips;  // [ntrip]
  const int* orbits;        // [norbits] packed A | B<<10 | C<<20, A <= B <= C
  const double* J;          // [nw*nw][v][v]   J_xy[u,w] = (xu|yw)
  const double* t1;         // [o][v]
  const double* eps_occ;    // [o]
  const double* eps_vir;    // [v]
  const double* t2;         // [o][o][v][v]   (Fock term only)
  const double* f_ov;       // [o][v] occupied-virtual Fock block, or NULL (canonical reference)
  double* partial;          // [ntrip][norbits]
  int ntrip, norbits, nbv, v, nw, use_t1, o;
};
int launch_energy(const EnergyArgs& a, cudaStream_t s);

// e_trip[trips[t].index] = weight(i,j,k) * sum_orbits partial[t][:]   (fixed order)
int launch_reduce_triplets(const double* partial, const TripletRec* trips, int ntrip, int norbits,
                           double* e_trip, cudaStream_t s);
// *out = sum_n e_trip[n] in a fixed order (single block)
int launch_final_sum(const double* e_trip, long long n, double* out, cudaStream_t s);

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
