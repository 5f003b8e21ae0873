// pack.cu — one-time repacking of the caller's arrays into the K-major, TMA-friendly layouts the
// tile-GEMM engine reads.  All HBM-bound, coalesced both ways.
#include "kernels.cuh"

namespace bqc {

// ---------------------------------------------------------------- [nq][in_pitch] -> [nr][qp] (zero pad)
// out[row(r)][q] = in[q][r0 + r], r < nr, q < nq; zero for nq <= q < qp.  row(r) = r, or, with perm_v > 0, the
// pair-transposed row: r0 + r = i * perm_v + a  ->  row = a * perm_o + i  (B_ov[Q,i,a] -> Bt_ov'[(a,i)][Q], the
// particle-hole dual used by the abc-driven schedule).
__global__ void transpose_pad_kernel(const double* __restrict__ in, long long in_pitch, long long r0,
                                     double* __restrict__ out, int nq, long long nr, int qp, int perm_v,
                                     int perm_o) {
  __shared__ double tile[32][33];
  const long long rb = (long long)blockIdx.x * 32;
  const int q0 = blockIdx.y * 32;
  for (int dy = threadIdx.y; dy < 32; dy += blockDim.y) {
    const int q = q0 + dy;
    const long long r = rb + threadIdx.x;
    tile[dy][threadIdx.x] = (q < nq && r < nr) ? in[(size_t)q * in_pitch + r0 + r] : 0.0;
  }
  __syncthreads();
  for (int dy = threadIdx.y; dy < 32; dy += blockDim.y) {
    const long long r = rb + dy;
    const int q = q0 + threadIdx.x;
    if (r < nr && q < qp) {
      long long row = r;
      if (perm_v > 0) {
        const long long c = r0 + r;
        row = (c % perm_v) * perm_o + c / perm_v;
      }
      out[(size_t)row * qp + q] = tile[threadIdx.x][dy];
    }
  }
}

int launch_transpose_pad(const double* in, long long in_pitch, long long r0, long long nr, double* out, int nq,
                         int qp, int perm_v, int perm_o, cudaStream_t s) {
  if (nr <= 0) return BQC_OK;
  dim3 grid((unsigned)((nr + 31) / 32), ceil_div(qp, 32));
  transpose_pad_kernel<<<grid, dim3(32, 8), 0, s>>>(in, in_pitch, r0, out, nq, nr, qp, perm_v, perm_o);
  count_launch();
  BQC_CUDA_OK(cudaGetLastError());
  return BQC_OK;
}

// ---------------------------------------------------------------- out[b][c][r] = scale * in[b][r][c]
// (the particle-hole dual arrays of the abc-driven schedule, t_energy.cu)
__global__ void transpose_scale_kernel(const double* __restrict__ in, double* __restrict__ out, long long nr,
                                       long long nc, double scale) {
  __shared__ double tile[32][33];
  const long long c0 = (long long)blockIdx.x * 32, r0 = (long long)blockIdx.y * 32;
  const double* src = in + (size_t)blockIdx.z * nr * nc;
  double* dst = out + (size_t)blockIdx.z * nr * nc;
  for (int dy = threadIdx.y; dy < 32; dy += blockDim.y) {
    const long long r = r0 + dy, c = c0 + threadIdx.x;
    tile[dy][threadIdx.x] = (r < nr && c < nc) ? src[r * nc + c] : 0.0;
  }
  __syncthreads();
  for (int dy = threadIdx.y; dy < 32; dy += blockDim.y) {
    const long long c = c0 + dy, r = r0 + threadIdx.x;
    if (c < nc && r < nr) dst[c * nr + r] = scale * tile[threadIdx.x][dy];
  }
}

int launch_transpose_scale(const double* in, double* out, int batch, long long nr, long long nc, double scale,
                           cudaStream_t s) {
  const long long gx = (nc + 31) / 32, gy = (nr + 31) / 32;
  if (batch <= 0 || nr <= 0 || nc <= 0) return BQC_OK;
  if (gy > 65535 || batch > 65535 || gx > 2147483647LL) {
    set_error(BQC_ERR_INVALID_SIZE, "transpose of %d x %lld x %lld exceeds the launch grid", batch, nr, nc);
    return BQC_ERR_INVALID_SIZE;
  }
  transpose_scale_kernel<<<dim3((unsigned)gx, (unsigned)gy, (unsigned)batch), dim3(32, 8), 0, s>>>(in, out, nr, nc,
                                                                                                   scale);
  count_launch();
  BQC_CUDA_OK(cudaGetLastError());
  return BQC_OK;
}

// ---------------------------------------------------------------- t2 rows -> particle columns of B~
// B~[(sz0 + z) * nslots + (sy0 + y)][r][d] = t2[z0 + z][y0 + y][r][d],  d < v  (row pitch kp; columns >= v untouched)
__global__ void btilde_t2_kernel(const double* __restrict__ t2, double* __restrict__ btil, int o, int v, int kp,
                                 int nslots, int z0, int y0, int ny, int sz0, int sy0) {
  // one block per (z, y, r) row
  const long long row = blockIdx.x;
  const int r = (int)(row % v);
  const int zy = (int)(row / v);
  const int z = zy / ny, y = zy % ny;
  const double* src = t2 + (((size_t)(z0 + z) * o + (y0 + y)) * v + r) * v;
  double* dst = btil + (((size_t)(sz0 + z) * nslots + (sy0 + y)) * v + r) * kp;
  for (int d = threadIdx.x; d < v; d += blockDim.x) dst[d] = src[d];
}

// abc-driven schedule (pipeline o = nvir, v = nocc; t2c = the caller's t2[nocc][nocc][nvir][nvir]):
// B~[(sz0+z) * nslots + (sy0+y)][r][d] = t2'[z0+z][y0+y][r][d] = -t2c[r][d][z0+z][y0+y]
// A 32 x 32 tile over (d, y) through shared memory: reads run along y, writes along d.
__global__ void btilde_t2_dual_kernel(const double* __restrict__ t2c, double* __restrict__ btil, int o, int v,
                                      int kp, int nslots, int z0, int y0, int ny, int sz0, int sy0) {
  __shared__ double tile[32][33];
  const int z = blockIdx.z / v, r = blockIdx.z % v;
  const int yb = blockIdx.x * 32, db = blockIdx.y * 32;
  const size_t o2 = (size_t)o * o;
  for (int dy = threadIdx.y; dy < 32; dy += blockDim.y) {
    const int d = db + dy, y = yb + threadIdx.x;
    tile[dy][threadIdx.x] =
        (d < v && y < ny) ? t2c[((size_t)r * v + d) * o2 + (size_t)(z0 + z) * o + (y0 + y)] : 0.0;
  }
  __syncthreads();
  for (int dy = threadIdx.y; dy < 32; dy += blockDim.y) {
    const int y = yb + dy, d = db + threadIdx.x;
    if (y < ny && d < v)
      btil[(((size_t)(sz0 + z) * nslots + (sy0 + y)) * v + r) * kp + d] = -tile[threadIdx.x][dy];
  }
}

int launch_btilde_t2(const double* t2, double* btil, int o, int v, int kp, int nslots, int z0, int nz, int y0,
                     int ny, int sz0, int sy0, bool dual, cudaStream_t s) {
  if (nz <= 0 || ny <= 0) return BQC_OK;
  if (!dual) {
    const long long rows = (long long)nz * ny * v;
    btilde_t2_kernel<<<(unsigned)rows, 128, 0, s>>>(t2, btil, o, v, kp, nslots, z0, y0, ny, sz0, sy0);
  } else {
    if ((long long)nz * v > 65535) {
      set_error(BQC_ERR_INVALID_SIZE, "B~ block of %d x %d rows exceeds the launch grid", nz, v);
      return BQC_ERR_INVALID_SIZE;
    }
    dim3 grid(ceil_div(ny, 32), ceil_div(v, 32), nz * v);
    btilde_t2_dual_kernel<<<grid, dim3(32, 8), 0, s>>>(t2, btil, o, v, kp, nslots, z0, y0, ny, sz0, sy0);
  }
  count_launch();
  BQC_CUDA_OK(cudaGetLastError());
  return BQC_OK;
}

// ---------------------------------------------------------------- hole columns of the slabs
// in  : t2[x][l][(p,q)]  (l rows of v^2)      out : slab[slot][(p,q)][v + l]  (pitch kp)
__global__ void slab_holes_kernel(const double* __restrict__ t2, double* __restrict__ slabs, int o, int v,
                                  int kp, int x0, int slot0) {
  __shared__ double tile[32][33];
  const int s = blockIdx.z;
  const size_t v2 = (size_t)v * v;
  const double* in = t2 + (size_t)(x0 + s) * o * v2;
  double* out = slabs + (size_t)(slot0 + s) * v2 * kp;
  const size_t pq0 = (size_t)blockIdx.x * 32;
  const int l0 = blockIdx.y * 32;
  for (int dy = threadIdx.y; dy < 32; dy += blockDim.y) {
    const int l = l0 + dy;
    const size_t pq = pq0 + threadIdx.x;
    tile[dy][threadIdx.x] = (l < o && pq < v2) ? in[(size_t)l * v2 + pq] : 0.0;
  }
  __syncthreads();
  for (int dy = threadIdx.y; dy < 32; dy += blockDim.y) {
    const size_t pq = pq0 + dy;
    const int l = l0 + threadIdx.x;
    if (pq < v2 && l < o) out[pq * kp + v + l] = -tile[threadIdx.x][dy];
  }
}

// abc-driven schedule: slab[slot][(p,q)][v + l] = -t2'[x][l][p][q] = +t2c[p][q][x][l]: a row copy
// (pipeline o = nvir rows of length o, one per (slot, p, q)).
__global__ void slab_holes_dual_kernel(const double* __restrict__ t2c, double* __restrict__ slabs, int o, int v,
                                       int kp, int x0, int slot0) {
  const size_t pq = blockIdx.x;
  const int s = blockIdx.y;
  const double* src = t2c + (pq * o + (size_t)(x0 + s)) * o;
  double* dst = slabs + ((size_t)(slot0 + s) * v * v + pq) * kp + v;
  for (int l = threadIdx.x; l < o; l += blockDim.x) dst[l] = src[l];
}

int launch_slab_holes(const double* t2, double* slabs, int o, int v, int kp, int x0, int nx, int slot0, bool dual,
                      cudaStream_t s) {
  if (nx <= 0) return BQC_OK;
  const size_t v2 = (size_t)v * v;
  if (!dual) {
    dim3 grid((unsigned)((v2 + 31) / 32), ceil_div(o, 32), nx);
    slab_holes_kernel<<<grid, dim3(32, 8), 0, s>>>(t2, slabs, o, v, kp, x0, slot0);
  } else {
    dim3 grid((unsigned)v2, nx);
    slab_holes_dual_kernel<<<grid, 128, 0, s>>>(t2, slabs, o, v, kp, x0, slot0);
  }
  count_launch();
  BQC_CUDA_OK(cudaGetLastError());
  return BQC_OK;
}

// ---------------------------------------------------------------- strided 3-D copy
__global__ void copy3_kernel(const double* __restrict__ in, long long sa, long long sb, long long sc,
                             double* __restrict__ out, int na, int nb, int nc) {
  const long long total = (long long)na * nb * nc;
  for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < total;
       e += (long long)gridDim.x * blockDim.x) {
    const int c = (int)(e % nc);
    const long long ab = e / nc;
    const int b = (int)(ab % nb);
    const long long a = ab / nb;
    out[e] = in[a * sa + b * sb + c * sc];
  }
}

int launch_copy3(const double* in, long long sa, long long sb, long long sc, double* out, int na, int nb,
                 int nc, cudaStream_t s) {
  const long long total = (long long)na * nb * nc;
  if (total <= 0) return BQC_OK;
  const int grid = (int)((total + 255) / 256 < 4096 ? (total + 255) / 256 : 4096);
  copy3_kernel<<<grid, 256, 0, s>>>(in, sa, sb, sc, out, na, nb, nc);
  count_launch();
  BQC_CUDA_OK(cudaGetLastError());
  return BQC_OK;
}

}  // namespace bqc
