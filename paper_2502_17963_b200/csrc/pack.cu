// pack.cu — one-time repacking of the caller's arrays into the K-major, TMA-friendly layouts the
// tile-GEMM engine reads.  All HBM-bound, coalesced both ways.
#include "kernels.cuh"

namespace bqc {

// ---------------------------------------------------------------- [nq][nr] -> [nr][qp] (zero pad)
__global__ void transpose_pad_kernel(const double* __restrict__ in, double* __restrict__ out, int nq,
                                     int nr, int qp) {
  __shared__ double tile[32][33];
  const int r0 = blockIdx.x * 32, q0 = blockIdx.y * 32;
  for (int dy = threadIdx.y; dy < 32; dy += blockDim.y) {
    const int q = q0 + dy, r = r0 + threadIdx.x;
    tile[dy][threadIdx.x] = (q < nq && r < nr) ? in[(size_t)q * nr + r] : 0.0;
  }
  __syncthreads();
  for (int dy = threadIdx.y; dy < 32; dy += blockDim.y) {
    const int r = r0 + dy, q = q0 + threadIdx.x;
    if (r < nr && q < qp) out[(size_t)r * qp + q] = tile[threadIdx.x][dy];
  }
}

int launch_transpose_pad(const double* in, double* out, int nq, int nr, int qp, cudaStream_t s) {
  dim3 grid(ceil_div(nr, 32), ceil_div(qp, 32));
  transpose_pad_kernel<<<grid, dim3(32, 8), 0, s>>>(in, out, nq, nr, qp);
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

// ---------------------------------------------------------------- t2 rows -> Btilde rows
__global__ void btilde_t2_kernel(const double* __restrict__ t2, double* __restrict__ btil, int o, int v,
                                 const int* __restrict__ act, int na, int kp) {
  // one block per (pair, r) row
  const long long row = blockIdx.x;
  const int r = (int)(row % v);
  const int pair = (int)(row / v);
  const int z = act[pair / na], y = act[pair % na];
  const double* src = t2 + (((size_t)z * o + y) * v + r) * v;
  double* dst = btil + (size_t)row * kp;
  for (int d = threadIdx.x; d < v; d += blockDim.x) dst[d] = src[d];
}

int launch_btilde_t2(const double* t2, double* btil, int o, int v, const int* act_dev, int na, int kp,
                     cudaStream_t s) {
  const long long rows = (long long)na * na * v;
  btilde_t2_kernel<<<(unsigned)rows, 128, 0, s>>>(t2, btil, o, v, act_dev, na, kp);
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

int launch_slab_holes(const double* t2, double* slabs, int o, int v, int kp, int x0, int nx,
                      int slot0, cudaStream_t s) {
  if (nx <= 0) return BQC_OK;
  const size_t v2 = (size_t)v * v;
  dim3 grid((unsigned)((v2 + 31) / 32), ceil_div(o, 32), nx);
  slab_holes_kernel<<<grid, dim3(32, 8), 0, s>>>(t2, slabs, o, v, kp, x0, slot0);
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
