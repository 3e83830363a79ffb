// init.cu — (f4) geometry-aware initialisation of the surfels from a DSM:
//   area-weighted sampling   weight of a DSM cell a = |dx x dy| = cell^2 sqrt(1 + h_x^2 + h_y^2) (finite differences:
//                            central inside, one-sided on the border), cumulative sum in double precision (three-phase
//                            device scan), inverse transform by binary search with the caller's uniform numbers;
//   centre                   jittered inside the cell and lifted to the cell's tangent plane;
//   orientation              n = (-h_x, -h_y, 1)/|.|, t_u = Gram-Schmidt of the world x axis against n, t_v = n x t_u,
//                            R = [t_u | t_v | n] -> quaternion (w >= 0);
//   scale                    mean distance to the 3 nearest other centres: uniform xy grid (counting sort of the points
//                            into cells), ring-by-ring search that stops once the third-best distance is inside the
//                            searched square (exact kNN).
// One-time work, HBM/latency-bound; none of it is on the per-iteration path.
#include "internal.cuh"

namespace satsplat {

constexpr int kScanItems = 4, kScanBlock = 1024, kScanChunk = kScanItems * kScanBlock;

__device__ __forceinline__ void dsm_slopes(const float* __restrict__ h, int W, int H, int col, int row, double inv_cell, double& hx,
                                           double& hy) {
  const int c0 = max(col - 1, 0), c1 = min(col + 1, W - 1), r0 = max(row - 1, 0), r1 = min(row + 1, H - 1);
  hx = c1 > c0 ? ((double)h[(size_t)row * W + c1] - (double)h[(size_t)row * W + c0]) * inv_cell / (double)(c1 - c0) : 0.0;
  hy = r1 > r0 ? ((double)h[(size_t)r1 * W + col] - (double)h[(size_t)r0 * W + col]) * inv_cell / (double)(r1 - r0) : 0.0;
}

__global__ void __launch_bounds__(256) dsm_weights_kernel(const float* __restrict__ h, int W, int H, double cell, double* __restrict__ w) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= (long long)W * H) return;
  double hx, hy;
  dsm_slopes(h, W, H, (int)(i % W), (int)(i / W), 1.0 / cell, hx, hy);
  w[i] = cell * cell * sqrt(1.0 + hx * hx + hy * hy);
}

// block-wide exclusive scan of one double per thread (1024 threads); returns the exclusive prefix, *total = block sum
__device__ __forceinline__ double block_scan_double(double v, double* s_warp, double* total) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  double inc = v;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const double t = __shfl_up_sync(0xffffffffu, inc, d);
    if (lane >= d) inc += t;
  }
  if (lane == 31) s_warp[warp] = inc;
  __syncthreads();
  if (warp == 0) {
    double w = s_warp[lane];
    double winc = w;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const double t = __shfl_up_sync(0xffffffffu, winc, d);
      if (lane >= d) winc += t;
    }
    s_warp[lane] = winc - w;          // exclusive over warps
    if (lane == 31) s_warp[32] = winc;
  }
  __syncthreads();
  const double r = s_warp[warp] + inc - v;
  *total = s_warp[32];
  __syncthreads();
  return r;
}

__global__ void __launch_bounds__(kScanBlock) cdf_partials_kernel(const double* __restrict__ w, long long M, double* __restrict__ partial) {
  __shared__ double s_warp[33];
  const long long base = (long long)blockIdx.x * kScanChunk + (long long)threadIdx.x * kScanItems;
  double s = 0.0;
#pragma unroll
  for (int k = 0; k < kScanItems; ++k)
    if (base + k < M) s += w[base + k];
  double total;
  block_scan_double(s, s_warp, &total);
  if (threadIdx.x == 0) partial[blockIdx.x] = total;
}

__global__ void __launch_bounds__(kScanBlock) cdf_top_kernel(double* __restrict__ partial, int nblocks, double* __restrict__ total_out) {
  __shared__ double s_warp[33];
  double carry = 0.0;
  for (int base = 0; base < nblocks; base += kScanBlock) {
    const int i = base + threadIdx.x;
    const double v = i < nblocks ? partial[i] : 0.0;
    double total;
    const double ex = block_scan_double(v, s_warp, &total);
    if (i < nblocks) partial[i] = carry + ex;      // exclusive prefix of the block sums
    carry += total;
  }
  if (threadIdx.x == 0) *total_out = carry;
}

__global__ void __launch_bounds__(kScanBlock) cdf_apply_kernel(double* __restrict__ w, long long M, const double* __restrict__ partial) {
  __shared__ double s_warp[33];
  const long long base = (long long)blockIdx.x * kScanChunk + (long long)threadIdx.x * kScanItems;
  double v[kScanItems], s = 0.0;
#pragma unroll
  for (int k = 0; k < kScanItems; ++k) {
    v[k] = base + k < M ? w[base + k] : 0.0;
    s += v[k];
  }
  double total;
  double run = partial[blockIdx.x] + block_scan_double(s, s_warp, &total);
#pragma unroll
  for (int k = 0; k < kScanItems; ++k) {
    run += v[k];
    if (base + k < M) w[base + k] = run;            // inclusive cumulative weight, in place
  }
}

__global__ void __launch_bounds__(256) init_sample_kernel(const float* __restrict__ h, int W, int H, double cell, double ox, double oy,
                                                          long long N, const float* __restrict__ u, const float* __restrict__ jx,
                                                          const float* __restrict__ jy, const double* __restrict__ cdf,
                                                          const double* __restrict__ total, float* __restrict__ means,
                                                          float* __restrict__ quats, int32_t* __restrict__ cells) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  const long long M = (long long)W * H;
  const double target = (double)u[i] * *total;
  long long lo = 0, hi = M - 1;                        // first index with cdf > target (clamped to the last cell)
  while (lo < hi) {
    const long long mid = (lo + hi) >> 1;
    if (cdf[mid] > target) hi = mid; else lo = mid + 1;
  }
  const int row = (int)(lo / W), col = (int)(lo % W);
  double hx, hy;
  dsm_slopes(h, W, H, col, row, 1.0 / cell, hx, hy);
  const double ax = (double)jx[i], ay = (double)jy[i];
  means[3 * i + 0] = (float)(ox + (col + ax) * cell);
  means[3 * i + 1] = (float)(oy + (row + ay) * cell);
  means[3 * i + 2] = (float)((double)h[(size_t)row * W + col] + hx * (ax - 0.5) * cell + hy * (ay - 0.5) * cell);
  if (cells) cells[i] = (int32_t)lo;
  // frame: n, t_u = normalise(e_x - (e_x.n) n), t_v = n x t_u
  const double inn = rsqrt(1.0 + hx * hx + hy * hy);
  const double n0 = -hx * inn, n1 = -hy * inn, n2 = inn;
  double t0 = 1.0 - n0 * n0, t1 = -n0 * n1, t2 = -n0 * n2;
  const double itn = rsqrt(t0 * t0 + t1 * t1 + t2 * t2);
  t0 *= itn; t1 *= itn; t2 *= itn;
  const double v0 = n1 * t2 - n2 * t1, v1 = n2 * t0 - n0 * t2, v2 = n0 * t1 - n1 * t0;
  // R = [t | v | n] (columns) -> quaternion (w, x, y, z), largest-pivot branch, w >= 0
  const double m00 = t0, m10 = t1, m20 = t2, m01 = v0, m11 = v1, m21 = v2, m02 = n0, m12 = n1, m22 = n2;
  const double tr = m00 + m11 + m22;
  double qw, qx, qy, qz;
  if (tr > 0) {
    const double s = sqrt(tr + 1.0) * 2;
    qw = 0.25 * s; qx = (m21 - m12) / s; qy = (m02 - m20) / s; qz = (m10 - m01) / s;
  } else if (m00 > m11 && m00 > m22) {
    const double s = sqrt(1.0 + m00 - m11 - m22) * 2;
    qw = (m21 - m12) / s; qx = 0.25 * s; qy = (m01 + m10) / s; qz = (m02 + m20) / s;
  } else if (m11 > m22) {
    const double s = sqrt(1.0 + m11 - m00 - m22) * 2;
    qw = (m02 - m20) / s; qx = (m01 + m10) / s; qy = 0.25 * s; qz = (m12 + m21) / s;
  } else {
    const double s = sqrt(1.0 + m22 - m00 - m11) * 2;
    qw = (m10 - m01) / s; qx = (m02 + m20) / s; qy = (m12 + m21) / s; qz = 0.25 * s;
  }
  const double sg = qw < 0 ? -1.0 : 1.0;
  reinterpret_cast<float4*>(quats)[i] = make_float4((float)(sg * qw), (float)(sg * qx), (float)(sg * qy), (float)(sg * qz));
}

// ---- kNN point spacing on a uniform xy grid ------------------------------------------------------------------
struct KnnGrid {
  float ox, oy, g, inv_g;   // origin and cell size of the grid
  int GX, GY;
};

__device__ __forceinline__ int grid_cell_x(const KnnGrid& G, float x) { return min(max((int)floorf((x - G.ox) * G.inv_g), 0), G.GX - 1); }
__device__ __forceinline__ int grid_cell_y(const KnnGrid& G, float y) { return min(max((int)floorf((y - G.oy) * G.inv_g), 0), G.GY - 1); }

__global__ void __launch_bounds__(256) knn_count_kernel(KnnGrid G, long long N, const float* __restrict__ means, uint32_t* __restrict__ count) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  atomicAdd(count + grid_cell_y(G, means[3 * i + 1]) * G.GX + grid_cell_x(G, means[3 * i]), 1u);
}

// exclusive scan of the cell counters (one CTA, chunked); the counters become the scatter cursors (zeroed)
__global__ void __launch_bounds__(1024) knn_scan_kernel(int ncells, uint32_t* __restrict__ count, uint32_t* __restrict__ start) {
  __shared__ uint32_t s_warp[33];
  uint32_t carry = 0;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (int base = 0; base < ncells; base += 1024) {
    const int i = base + threadIdx.x;
    const uint32_t v = i < ncells ? count[i] : 0u;
    uint32_t inc = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const uint32_t t = __shfl_up_sync(0xffffffffu, inc, d);
      if (lane >= d) inc += t;
    }
    if (lane == 31) s_warp[warp] = inc;
    __syncthreads();
    if (warp == 0) {
      const uint32_t w = s_warp[lane];
      uint32_t winc = w;
#pragma unroll
      for (int d = 1; d < 32; d <<= 1) {
        const uint32_t t = __shfl_up_sync(0xffffffffu, winc, d);
        if (lane >= d) winc += t;
      }
      s_warp[lane] = winc - w;
      if (lane == 31) s_warp[32] = winc;
    }
    __syncthreads();
    if (i < ncells) {
      start[i] = carry + s_warp[warp] + inc - v;
      count[i] = 0u;
    }
    carry += s_warp[32];
    __syncthreads();
  }
  if (threadIdx.x == 0) start[ncells] = carry;
}

__global__ void __launch_bounds__(256) knn_scatter_kernel(KnnGrid G, long long N, const float* __restrict__ means,
                                                          const uint32_t* __restrict__ start, uint32_t* __restrict__ cursor,
                                                          uint32_t* __restrict__ sorted) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  const int c = grid_cell_y(G, means[3 * i + 1]) * G.GX + grid_cell_x(G, means[3 * i]);
  sorted[start[c] + atomicAdd(cursor + c, 1u)] = (uint32_t)i;
}

__global__ void __launch_bounds__(128) knn_scale_kernel(KnnGrid G, long long N, float fallback, const float* __restrict__ means,
                                                        const uint32_t* __restrict__ start, const uint32_t* __restrict__ sorted,
                                                        float* __restrict__ scales) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  float s = fallback;
  if (N > 3) {
    const float px = means[3 * i], py = means[3 * i + 1], pz = means[3 * i + 2];
    const int cx = grid_cell_x(G, px), cy = grid_cell_y(G, py);
    float b0 = 3.0e38f, b1 = 3.0e38f, b2 = 3.0e38f;   // three smallest squared distances, ascending
    const int rmax = max(max(cx, G.GX - 1 - cx), max(cy, G.GY - 1 - cy));
    auto visit = [&](int xx, int yy) {
      if (xx < 0 || xx >= G.GX || yy < 0 || yy >= G.GY) return;
      const int c = yy * G.GX + xx;
      for (uint32_t k = start[c]; k < start[c + 1]; ++k) {
        const uint32_t j = sorted[k];
        if ((long long)j == i) continue;
        const float dx = means[3 * j] - px, dy = means[3 * j + 1] - py, dz = means[3 * j + 2] - pz;
        const float d = dx * dx + dy * dy + dz * dz;
        if (d < b2) {
          if (d < b1) { b2 = b1; if (d < b0) { b1 = b0; b0 = d; } else b1 = d; } else b2 = d;
        }
      }
    };
    for (int r = 0; r <= rmax; ++r) {
      const int y0 = cy - r, y1 = cy + r, x0 = cx - r, x1 = cx + r;
      // the cells at Chebyshev distance exactly r: top and bottom rows in full, left and right columns in between
      for (int xx = x0; xx <= x1; ++xx) {
        visit(xx, y0);
        if (r > 0) visit(xx, y1);
      }
      for (int yy = y0 + 1; yy < y1; ++yy) {
        visit(x0, yy);
        visit(x1, yy);
      }
      // everything outside the searched square is at least `reach` away (in xy, hence in 3-D)
      const float reach = fminf(fminf(px - (G.ox + (float)x0 * G.g), G.ox + (float)(x1 + 1) * G.g - px),
                                fminf(py - (G.oy + (float)y0 * G.g), G.oy + (float)(y1 + 1) * G.g - py));
      if (b2 < 3.0e38f && reach > 0.f && b2 <= reach * reach) break;
    }
    s = (sqrtf(b0) + sqrtf(b1) + sqrtf(b2)) * (1.0f / 3.0f);
  }
  scales[2 * i] = s;
  scales[2 * i + 1] = s;
}

// in-place inclusive cumulative sum of M doubles (three launches); partial needs M / 4096 + 9 doubles, total = partial + nb
int64_t cdf_scan_partials(int64_t M) { return (M + kScanChunk - 1) / kScanChunk + 9; }
cudaError_t launch_cdf_scan(double* w, long long M, double* partial, double** total_out, cudaStream_t s) {
  const int nb = (int)((M + kScanChunk - 1) / kScanChunk);
  *total_out = partial + nb;
  g_kernel_launches += 3;
  cdf_partials_kernel<<<nb, kScanBlock, 0, s>>>(w, M, partial);
  cdf_top_kernel<<<1, kScanBlock, 0, s>>>(partial, nb, partial + nb);
  cdf_apply_kernel<<<nb, kScanBlock, 0, s>>>(w, M, partial);
  return cudaGetLastError();
}

int64_t init_scratch_bytes(int W, int H, int64_t N) {
  const int64_t M = (int64_t)W * H;
  const int64_t nb = (M + kScanChunk - 1) / kScanChunk;
  const int64_t cells = N / 2 + 1024;                    // upper bound of the kNN grid (about N / 4 cells are used)
  return M * 8 + (nb + 8) * 8 + (cells + 1) * 4 * 2 + N * 4 + 256;
}

cudaError_t launch_init_from_dsm(const float* dsm, int W, int H, float cell, float ox, float oy, int64_t N, const float* u,
                                 const float* jx, const float* jy, void* scratch, float* means, float* quats, float* scales,
                                 int32_t* cells_out, cudaStream_t s) {
  if (N == 0) return cudaSuccess;
  const long long M = (long long)W * H;
  const int nb = (int)((M + kScanChunk - 1) / kScanChunk);
  char* p = reinterpret_cast<char*>(scratch);
  double* cdf = reinterpret_cast<double*>(p);           p += M * 8;
  double* partial = reinterpret_cast<double*>(p);       p += ((int64_t)nb + 8) * 8;   // [nb] + total at [nb]
  double* total = partial + nb;
  // kNN grid: about four points per cell on flat ground, never finer than the DSM
  KnnGrid G;
  const double ext_x = (double)W * cell, ext_y = (double)H * cell;
  double g = 2.0 * sqrt(ext_x * ext_y / (double)N);
  if (g < cell) g = cell;
  G.GX = (int)ceil(ext_x / g); G.GY = (int)ceil(ext_y / g);
  if (G.GX < 1) G.GX = 1;
  if (G.GY < 1) G.GY = 1;
  while ((int64_t)G.GX * G.GY > N / 2 + 1024) { g *= 1.5; G.GX = (int)ceil(ext_x / g); G.GY = (int)ceil(ext_y / g); }
  G.ox = ox; G.oy = oy; G.g = (float)g; G.inv_g = (float)(1.0 / g);
  const int ncells = G.GX * G.GY;
  uint32_t* count = reinterpret_cast<uint32_t*>(p);     p += ((int64_t)N / 2 + 1024 + 1) * 4;
  uint32_t* start = reinterpret_cast<uint32_t*>(p);     p += ((int64_t)N / 2 + 1024 + 1) * 4;
  uint32_t* sorted = reinterpret_cast<uint32_t*>(p);
  cudaError_t e = cudaMemsetAsync(count, 0, (size_t)ncells * 4, s);
  if (e != cudaSuccess) return e;
  g_kernel_launches += 8;
  dsm_weights_kernel<<<(int)((M + 255) / 256), 256, 0, s>>>(dsm, W, H, (double)cell, cdf);
  cdf_partials_kernel<<<nb, kScanBlock, 0, s>>>(cdf, M, partial);
  cdf_top_kernel<<<1, kScanBlock, 0, s>>>(partial, nb, total);
  cdf_apply_kernel<<<nb, kScanBlock, 0, s>>>(cdf, M, partial);
  const int nbN = (int)((N + 255) / 256);
  init_sample_kernel<<<nbN, 256, 0, s>>>(dsm, W, H, (double)cell, (double)ox, (double)oy, N, u, jx, jy, cdf, total, means, quats, cells_out);
  knn_count_kernel<<<nbN, 256, 0, s>>>(G, N, means, count);
  knn_scan_kernel<<<1, 1024, 0, s>>>(ncells, count, start);
  knn_scatter_kernel<<<nbN, 256, 0, s>>>(G, N, means, start, count, sorted);
  ++g_kernel_launches;
  knn_scale_kernel<<<(int)((N + 127) / 128), 128, 0, s>>>(G, N, cell, means, start, sorted, scales);
  return cudaGetLastError();
}

}  // namespace satsplat
