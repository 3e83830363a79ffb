// binning.cu — (a2) exclusive scan of tile counts, key duplication, stable LSD radix sort of
// (tile id << 32 | depth bits) keys with surfel-id payloads, and per-tile range detection (PAPER.md:140:
// "sorted based on the depth of their centers and organized into tiles").  Integer work: bit-exact.
//
// No host synchronisation anywhere: K (the number of duplicated keys) lives in device memory, every kernel
// below runs on a fixed grid and reads K itself.  All stages are HBM/L2-bandwidth bound.
#include "internal.cuh"

namespace satsplat {

// ------------------------------------------------------------------------------------------------------------
// exclusive scan of count[N] -> offset[N+1]; three small kernels (block sums, top-level scan, apply)
// ------------------------------------------------------------------------------------------------------------
constexpr int kScanThreads = 256;
constexpr int kScanItems = 16;
constexpr int kScanTile = kScanThreads * kScanItems;  // 4096

__device__ __forceinline__ uint32_t warp_inclusive_scan(uint32_t v, int lane) {
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const uint32_t t = __shfl_up_sync(0xffffffffu, v, d);
    if (lane >= d) v += t;
  }
  return v;
}

// block-wide exclusive scan of one value per thread (256 threads); returns exclusive prefix, total in *total
__device__ __forceinline__ uint32_t block_exclusive_scan(uint32_t v, uint32_t* s_warp, uint32_t* total) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint32_t inc = warp_inclusive_scan(v, lane);
  if (lane == 31) s_warp[warp] = inc;
  __syncthreads();
  if (warp == 0) {
    const uint32_t w = lane < (int)(blockDim.x >> 5) ? s_warp[lane] : 0u;
    const uint32_t wi = warp_inclusive_scan(w, lane);
    s_warp[lane] = wi - w;
    if (lane == 31) s_warp[32] = wi;
  }
  __syncthreads();
  const uint32_t res = s_warp[warp] + inc - v;
  *total = s_warp[32];
  __syncthreads();
  return res;
}

__global__ void __launch_bounds__(kScanThreads) scan_block_sums_kernel(int N, const uint32_t* __restrict__ count,
                                                                       uint32_t* __restrict__ block_sums) {
  __shared__ uint32_t s_warp[33];
  const int base = blockIdx.x * kScanTile;
  uint32_t sum = 0;
#pragma unroll
  for (int k = 0; k < kScanItems; ++k) {
    const int i = base + k * kScanThreads + threadIdx.x;
    if (i < N) sum += count[i];
  }
  uint32_t total;
  block_exclusive_scan(sum, s_warp, &total);
  if (threadIdx.x == 0) block_sums[blockIdx.x] = total;
}

__global__ void __launch_bounds__(1024) scan_top_kernel(int nblocks, uint32_t* __restrict__ block_sums, Status* status,
                                                         uint32_t capacity) {
  __shared__ uint32_t s_warp[33];
  __shared__ unsigned long long s_big[32];
  // one block; each thread owns a contiguous chunk
  const int per = (nblocks + 1023) / 1024;
  const int b0 = threadIdx.x * per;
  uint32_t sum = 0;
  unsigned long long sum64 = 0;   // the grand total in 64 bits: a sum beyond 2^32 must be flagged, not wrapped
  for (int k = 0; k < per; ++k)
    if (b0 + k < nblocks) { sum += block_sums[b0 + k]; sum64 += block_sums[b0 + k]; }
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) sum64 += __shfl_xor_sync(0xffffffffu, sum64, d);
  if ((threadIdx.x & 31) == 0) s_big[threadIdx.x >> 5] = sum64;
  uint32_t total;
  uint32_t run = block_exclusive_scan(sum, s_warp, &total);   // (contains the barriers that publish s_big)
  for (int k = 0; k < per; ++k)
    if (b0 + k < nblocks) {
      const uint32_t v = block_sums[b0 + k];
      block_sums[b0 + k] = run;
      run += v;
    }
  if (threadIdx.x == 0) {
    unsigned long long t64 = 0;
    for (int w = 0; w < 32; ++w) t64 += s_big[w];
    status->K = t64 > 0xffffffffull ? 0xffffffffu : (uint32_t)t64;
    status->overflow = t64 > (unsigned long long)capacity ? 1u : 0u;
  }
}

__global__ void __launch_bounds__(kScanThreads) scan_apply_kernel(int N, const uint32_t* __restrict__ count,
                                                                  const uint32_t* __restrict__ block_sums,
                                                                  uint32_t* __restrict__ offset) {
  __shared__ uint32_t s_warp[33];
  // blocked arrangement: thread t owns items [t*16, t*16+16) of the tile so that a single block scan suffices
  const int base = blockIdx.x * kScanTile + threadIdx.x * kScanItems;
  uint32_t v[kScanItems];
  uint32_t sum = 0;
#pragma unroll
  for (int k = 0; k < kScanItems; k += 4) {
    if (base + k + 3 < N) {
      const uint4 t = *reinterpret_cast<const uint4*>(count + base + k);
      v[k] = t.x; v[k + 1] = t.y; v[k + 2] = t.z; v[k + 3] = t.w;
    } else {
#pragma unroll
      for (int j = 0; j < 4; ++j) v[k + j] = (base + k + j < N) ? count[base + k + j] : 0u;
    }
  }
#pragma unroll
  for (int k = 0; k < kScanItems; ++k) sum += v[k];
  uint32_t total;
  uint32_t run = block_exclusive_scan(sum, s_warp, &total) + block_sums[blockIdx.x];
#pragma unroll
  for (int k = 0; k < kScanItems; ++k) {
    if (base + k < N) offset[base + k] = run;
    run += v[k];
  }
  if (base <= N - 1 && base + kScanItems > N - 1) offset[N] = run;  // total after the last element
}

cudaError_t launch_scan(satsplat_ctx* c, int64_t N, cudaStream_t s) {
  const int nblocks = (int)((N + kScanTile - 1) / kScanTile);
  if (nblocks == 0) {
    const cudaError_t e = cudaMemsetAsync(c->status, 0, sizeof(Status), s);
    return e != cudaSuccess ? e : cudaMemsetAsync(c->offset, 0, sizeof(uint32_t), s);
  }
  g_kernel_launches += 3;
  scan_block_sums_kernel<<<nblocks, kScanThreads, 0, s>>>((int)N, c->count, c->block_sums);
  scan_top_kernel<<<1, 1024, 0, s>>>(nblocks, c->block_sums, c->status, (uint32_t)c->max_dup);
  scan_apply_kernel<<<nblocks, kScanThreads, 0, s>>>((int)N, c->count, c->block_sums, c->offset);
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------------------
// key duplication: surfel i writes count[i] keys (row-major over its tile rect) at offset[i].  One warp per 32
// surfels; surfels with many tiles are expanded cooperatively by the whole warp so that no thread serialises a
// 4000-tile splat (oversized Gaussians).
// ------------------------------------------------------------------------------------------------------------
constexpr int kDupCoopThreshold = 16;

__global__ void __launch_bounds__(256) duplicate_kernel(int N, int TX, const ushort4* __restrict__ rect,
                                                        const uint32_t* __restrict__ count,
                                                        const uint32_t* __restrict__ offset,
                                                        const uint32_t* __restrict__ depth_key, uint64_t* __restrict__ keys,
                                                        uint32_t* __restrict__ vals, uint32_t capacity) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int lane = threadIdx.x & 31;
  uint32_t cnt = 0, off = 0, dk = 0;
  ushort4 r = make_ushort4(0, 0, 0, 0);
  if (i < N) {
    cnt = count[i];
    if (cnt) { off = offset[i]; dk = depth_key[i]; r = rect[i]; }
  }
  if (cnt && off + cnt > capacity) cnt = 0;  // overflow: flagged by the scan, nothing written out of bounds
  // small splats: the owning thread writes them
  if (cnt && cnt <= kDupCoopThreshold) {
    uint32_t o = off;
    for (int ty = r.y; ty < r.w; ++ty)
      for (int tx = r.x; tx < r.z; ++tx) {
        keys[o] = ((uint64_t)(uint32_t)(ty * TX + tx) << 32) | dk;
        vals[o] = (uint32_t)i;
        ++o;
      }
  }
  // large splats: whole warp, coalesced
  unsigned big = __ballot_sync(0xffffffffu, cnt > kDupCoopThreshold);
  while (big) {
    const int src = __ffs(big) - 1;
    big &= big - 1;
    const uint32_t c2 = __shfl_sync(0xffffffffu, cnt, src);
    const uint32_t o2 = __shfl_sync(0xffffffffu, off, src);
    const uint32_t k2 = __shfl_sync(0xffffffffu, dk, src);
    const int x0 = __shfl_sync(0xffffffffu, (int)r.x, src), y0 = __shfl_sync(0xffffffffu, (int)r.y, src);
    const int x1 = __shfl_sync(0xffffffffu, (int)r.z, src);
    const int id = (blockIdx.x * blockDim.x + (threadIdx.x & ~31)) + src;
    const int w = x1 - x0;
    for (uint32_t e = lane; e < c2; e += 32) {
      const int ty = y0 + (int)(e / (uint32_t)w), tx = x0 + (int)(e % (uint32_t)w);
      keys[o2 + e] = ((uint64_t)(uint32_t)(ty * TX + tx) << 32) | k2;
      vals[o2 + e] = (uint32_t)id;
    }
  }
}

cudaError_t launch_duplicate(satsplat_ctx* c, int64_t N, cudaStream_t s) {
  if (N == 0) return cudaSuccess;
  ++g_kernel_launches;
  duplicate_kernel<<<(int)((N + 255) / 256), 256, 0, s>>>((int)N, c->cam.TX, reinterpret_cast<const ushort4*>(c->rect),
                                                          c->count, c->offset, c->depth_key, c->keys[0], c->vals[0],
                                                          (uint32_t)c->max_dup);
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------------------
// stable LSD radix sort, 8 bits per pass, 64-bit keys + 32-bit payloads.  Per pass: (1) per-block digit
// histogram over the block's contiguous chunk, (2) exclusive scan of the [digit][block] table, (3) stable
// scatter (ranks from warp match + per-warp counters).  Chunks are contiguous and processed in order, so the
// sort is stable; only as many passes as the key has significant bits (32 depth bits + ceil(log2 tiles)).
// ------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void sort_chunk(uint32_t K, uint32_t& begin, uint32_t& end) {
  const uint32_t tiles = (K + kSortTile - 1) / kSortTile;
  const uint32_t per = (tiles + gridDim.x - 1) / gridDim.x;
  begin = min((uint32_t)blockIdx.x * per * kSortTile, K);
  end = min(begin + per * kSortTile, K);
}

__global__ void __launch_bounds__(kSortThreads) sort_hist_kernel(const Status* __restrict__ status, uint32_t capacity,
                                                                 const uint64_t* __restrict__ keys, int shift,
                                                                 uint32_t* __restrict__ hist) {
  __shared__ uint32_t s_hist[256];
  const uint32_t K = min(status->K, capacity);
  uint32_t begin, end;
  sort_chunk(K, begin, end);
  s_hist[threadIdx.x] = 0;
  __syncthreads();
  const int lane = threadIdx.x & 31;
  for (uint32_t base = begin; base < end; base += kSortThreads) {
    const uint32_t i = base + threadIdx.x;
    const bool valid = i < end;
    const uint32_t d = valid ? (uint32_t)(keys[i] >> shift) & 255u : (256u + lane);
    const unsigned m = __match_any_sync(0xffffffffu, d);
    if (valid && lane == __ffs(m) - 1) atomicAdd(&s_hist[d], __popc(m));
  }
  __syncthreads();
  hist[threadIdx.x * gridDim.x + blockIdx.x] = s_hist[threadIdx.x];
}

// exclusive scan of the [digit][block] table (n = 256 * kSortBlocks entries) by ONE 1024-thread CTA with coalesced
// accesses: warp w owns the contiguous segment [w*seg, (w+1)*seg) and walks it 32 entries at a time.
__global__ void __launch_bounds__(1024) sort_scan_kernel(int n, uint32_t* __restrict__ hist) {
  __shared__ uint32_t s_warp[33];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int seg = ((n + 31) / 32 + 31) / 32 * 32;   // per-warp segment, multiple of 32
  const int begin = warp * seg, end = min(begin + seg, n);
  uint32_t sum = 0;
  for (int i = begin + lane; i < end; i += 32) sum += hist[i];
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, d);
  if (lane == 0) s_warp[warp] = sum;
  __syncthreads();
  if (warp == 0) {
    const uint32_t w = s_warp[lane];
    const uint32_t wi = warp_inclusive_scan(w, lane);
    s_warp[lane] = wi - w;
  }
  __syncthreads();
  uint32_t run = s_warp[warp];
  for (int i0 = begin; i0 < end; i0 += 32) {
    const int i = i0 + lane;
    const uint32_t v = i < end ? hist[i] : 0u;
    const uint32_t inc = warp_inclusive_scan(v, lane);
    if (i < end) hist[i] = run + inc - v;
    run += __shfl_sync(0xffffffffu, inc, 31);
  }
}

__global__ void __launch_bounds__(kSortThreads) sort_scatter_kernel(const Status* __restrict__ status, uint32_t capacity,
                                                                    const uint64_t* __restrict__ keys_in,
                                                                    const uint32_t* __restrict__ vals_in,
                                                                    uint64_t* __restrict__ keys_out,
                                                                    uint32_t* __restrict__ vals_out, int shift,
                                                                    const uint32_t* __restrict__ hist) {
  constexpr int kWarps = kSortThreads / 32;
  __shared__ uint32_t s_warp_hist[kWarps][256];
  __shared__ uint32_t s_base[256];       // running global base of each digit for this block
  __shared__ uint32_t s_tile_base[256];  // base of each digit for the current tile
  const uint32_t K = min(status->K, capacity);
  uint32_t begin, end;
  sort_chunk(K, begin, end);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const unsigned lt = (1u << lane) - 1u;
  s_base[threadIdx.x] = hist[threadIdx.x * gridDim.x + blockIdx.x];
  for (uint32_t tile = begin; tile < end; tile += kSortTile) {
#pragma unroll
    for (int w = 0; w < kWarps; ++w) s_warp_hist[w][threadIdx.x] = 0;
    __syncthreads();
    uint64_t key[kSortItems];
    uint32_t val[kSortItems], rank[kSortItems];
    const uint32_t wbase = tile + warp * (kSortItems * 32);
#pragma unroll
    for (int j = 0; j < kSortItems; ++j) {
      const uint32_t i = wbase + j * 32 + lane;
      const bool valid = i < end;
      key[j] = valid ? keys_in[i] : 0ull;
      val[j] = valid ? vals_in[i] : 0u;
    }
#pragma unroll
    for (int j = 0; j < kSortItems; ++j) {
      const uint32_t i = wbase + j * 32 + lane;
      const bool valid = i < end;
      const uint32_t d = valid ? (uint32_t)(key[j] >> shift) & 255u : (256u + lane);
      const unsigned m = __match_any_sync(0xffffffffu, d);
      uint32_t prev = 0;
      if (valid) prev = s_warp_hist[warp][d];
      __syncwarp();
      rank[j] = prev + __popc(m & lt);
      if (valid && lane == __ffs(m) - 1) s_warp_hist[warp][d] = prev + __popc(m);
      __syncwarp();
    }
    __syncthreads();
    {  // per digit: exclusive scan over the warps, then advance the running base
      const int d = threadIdx.x;
      uint32_t run = 0;
#pragma unroll
      for (int w = 0; w < kWarps; ++w) {
        const uint32_t c = s_warp_hist[w][d];
        s_warp_hist[w][d] = run;
        run += c;
      }
      const uint32_t b = s_base[d];
      s_tile_base[d] = b;
      s_base[d] = b + run;
    }
    __syncthreads();
#pragma unroll
    for (int j = 0; j < kSortItems; ++j) {
      const uint32_t i = wbase + j * 32 + lane;
      if (i < end) {
        const uint32_t d = (uint32_t)(key[j] >> shift) & 255u;
        const uint32_t dst = s_tile_base[d] + s_warp_hist[warp][d] + rank[j];
        keys_out[dst] = key[j];
        vals_out[dst] = val[j];
      }
    }
    __syncthreads();
  }
}

cudaError_t launch_sort(satsplat_ctx* c, cudaStream_t s) {
  const int tiles = c->cam.TX * c->cam.TY;
  int tile_bits = 0;
  while ((1 << tile_bits) < tiles) ++tile_bits;
  const int passes = (32 + tile_bits + 7) / 8;
  int cur = 0;
  for (int p = 0; p < passes; ++p) {
    const int shift = 8 * p;
    g_kernel_launches += 3;
    sort_hist_kernel<<<kSortBlocks, kSortThreads, 0, s>>>(c->status, (uint32_t)c->max_dup, c->keys[cur], shift, c->hist);
    sort_scan_kernel<<<1, 1024, 0, s>>>(256 * kSortBlocks, c->hist);
    sort_scatter_kernel<<<kSortBlocks, kSortThreads, 0, s>>>(c->status, (uint32_t)c->max_dup, c->keys[cur], c->vals[cur],
                                                            c->keys[cur ^ 1], c->vals[cur ^ 1], shift, c->hist);
    cur ^= 1;
  }
  c->sorted = cur;
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------------------
// tile ranges: ranges[t] = [first, last+1) of tile t in the sorted keys, (0,0) for empty tiles
// ------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) ranges_kernel(const Status* __restrict__ status, uint32_t capacity,
                                                     const uint64_t* __restrict__ keys, uint32_t* __restrict__ ranges) {
  const uint32_t K = min(status->K, capacity);
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < K; i += gridDim.x * blockDim.x) {
    const uint32_t t = (uint32_t)(keys[i] >> 32);
    if (i == 0 || (uint32_t)(keys[i - 1] >> 32) != t) ranges[2 * t] = i;
    if (i == K - 1 || (uint32_t)(keys[i + 1] >> 32) != t) ranges[2 * t + 1] = i + 1;
  }
}

cudaError_t launch_ranges(satsplat_ctx* c, cudaStream_t s) {
  const int tiles = c->cam.TX * c->cam.TY;
  const cudaError_t e = cudaMemsetAsync(c->ranges, 0, sizeof(uint32_t) * 2 * (size_t)tiles, s);
  if (e != cudaSuccess) return e;
  ++g_kernel_launches;
  ranges_kernel<<<c->sm_count * 8, 256, 0, s>>>(c->status, (uint32_t)c->max_dup, c->keys[c->sorted], c->ranges);
  return cudaGetLastError();
}

// ============================================================================================================
// Tile-sort binning (default mode): the same unique result as the stable radix sort above — entries ordered by
// (tile id, depth bits, surfel id) — but built the way the data wants on B200: the (tile, surfel) pairs of one
// view (2 M at C3) sit in L2, so instead of 6 full radix passes we
//   1. count pairs per tile with fire-and-forget RED atomics (fused into the preprocess kernel),
//   2. exclusive-scan the per-tile counts (this IS the tile-range table),
//   3. scatter (depth bits << 32 | surfel id) entries into their tile's segment in arrival order,
//   4. sort every segment in shared memory by the 64-bit (depth, id) composite, one warp per tile.
// Arrival order is nondeterministic, the sorted result is not: (depth, id) is a total order and each surfel occurs
// at most once per tile.  4 launches instead of 25, ~10x less traffic.
// ============================================================================================================

// Exclusive scan of tile_count[tiles] in two multi-CTA kernels (a single CTA took 18 us for the 64 KB of a 2048^2 view):
//  A. every CTA scans its 2048 counters (8 per thread, loaded as two uint4) and leaves the CTA-local exclusive prefix in
//     tile_start and its total in block_sums;
//  B. every CTA adds the totals of the CTAs before it (a handful of values), writes the tile ranges (= the scan), turns
//     the counters into scatter cursors that start at the tile's first position, and files the long lists on the
//     worklists of the mid / large sort kernels.  K and the overflow flag come from the 64-bit grand total.
constexpr int kTileScanThreads = 256;
constexpr int kTileScanItems = 8;
constexpr int kTileScanChunk = kTileScanThreads * kTileScanItems;   // 2048 tiles per CTA
#ifndef SATSPLAT_SORT_SMALL_MAX
#define SATSPLAT_SORT_SMALL_MAX 256
#endif
constexpr int kTileSortSmallMax = SATSPLAT_SORT_SMALL_MAX;    // entries one warp sorts in registers in the small-tile kernel (4 or 8 per lane)
constexpr int kTileSortMergeMax = 1024;   // entries the 4-warp merge kernel handles (4 runs of <= 256)
constexpr int kTileSortMerge16Max = 4096; // entries the 16-warp merge kernel handles (16 runs of <= 256)

__global__ void __launch_bounds__(kTileScanThreads) tile_scan_partial_kernel(int tiles, const uint32_t* __restrict__ tile_count,
                                                                             uint32_t* __restrict__ tile_start,
                                                                             uint32_t* __restrict__ block_sums,
                                                                             uint32_t* __restrict__ wl_count) {
  __shared__ uint32_t s_warp[33];
  if (blockIdx.x == 0 && threadIdx.x < 4) wl_count[threadIdx.x] = 0u;   // worklist lengths / cursors of this pass
  const int i0 = blockIdx.x * kTileScanChunk + threadIdx.x * kTileScanItems;
  uint32_t v[kTileScanItems];
  if (kCtrStride == 1 && i0 + kTileScanItems <= tiles) {
    const uint4 a = reinterpret_cast<const uint4*>(tile_count + i0)[0], b = reinterpret_cast<const uint4*>(tile_count + i0)[1];
    v[0] = a.x; v[1] = a.y; v[2] = a.z; v[3] = a.w; v[4] = b.x; v[5] = b.y; v[6] = b.z; v[7] = b.w;
  } else {
#pragma unroll
    for (int k = 0; k < kTileScanItems; ++k) v[k] = i0 + k < tiles ? tile_count[(size_t)(i0 + k) * kCtrStride] : 0u;
  }
  uint32_t part = 0;
#pragma unroll
  for (int k = 0; k < kTileScanItems; ++k) part += v[k];
  uint32_t total;
  uint32_t run = block_exclusive_scan(part, s_warp, &total);
#pragma unroll
  for (int k = 0; k < kTileScanItems; ++k) {
    if (i0 + k < tiles) tile_start[i0 + k] = run;
    run += v[k];
  }
  if (threadIdx.x == 0) block_sums[blockIdx.x] = total;
}

__global__ void __launch_bounds__(kTileScanThreads) tile_scan_finish_kernel(int tiles, int nblocks, uint32_t* __restrict__ cursor,
                                                                            const uint32_t* __restrict__ tile_start,
                                                                            const uint32_t* __restrict__ block_sums,
                                                                            uint32_t* __restrict__ ranges, Status* status,
                                                                            uint32_t capacity, uint32_t* __restrict__ wl_count,
                                                                            uint32_t* __restrict__ worklist) {
  // one tile per thread; this CTA's tiles lie inside chunk `cb` of kernel A
  __shared__ unsigned long long s_red[2][kTileScanThreads / 32];
  __shared__ unsigned long long s_off[2];
  const int i = blockIdx.x * kTileScanThreads + threadIdx.x;
  const int cb = (blockIdx.x * kTileScanThreads) / kTileScanChunk;
  // offset of the chunk = sum of the chunk totals before it; grand total in 64 bits (it may exceed 2^32: flagged as overflow)
  unsigned long long before = 0, all = 0;
  for (int b = threadIdx.x; b < nblocks; b += kTileScanThreads) {
    const unsigned long long t = block_sums[b];
    all += t;
    if (b < cb) before += t;
  }
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) {
    before += __shfl_xor_sync(0xffffffffu, before, d);
    all += __shfl_xor_sync(0xffffffffu, all, d);
  }
  if ((threadIdx.x & 31) == 0) { s_red[0][threadIdx.x >> 5] = before; s_red[1][threadIdx.x >> 5] = all; }
  __syncthreads();
  if (threadIdx.x == 0) {
    unsigned long long a = 0, b = 0;
    for (int w = 0; w < kTileScanThreads / 32; ++w) { a += s_red[0][w]; b += s_red[1][w]; }
    s_off[0] = a; s_off[1] = b;
  }
  __syncthreads();
  const unsigned long long total = s_off[1];
  const bool overflow = total > (unsigned long long)capacity;
  const uint32_t off = (uint32_t)s_off[0];
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    status->K = total > 0xffffffffull ? 0xffffffffu : (uint32_t)total;
    status->overflow = overflow ? 1u : 0u;
  }
  const int lane = threadIdx.x & 31;
  uint32_t len = 0;
  if (i < tiles) {
    const bool last_of_chunk = (i + 1 == tiles) || ((i + 1) % kTileScanChunk == 0);
    const uint32_t st = off + tile_start[i];
    const uint32_t en = off + (last_of_chunk ? block_sums[cb] : tile_start[i + 1]);
    const bool empty = en == st || overflow;         // overflow: nothing is rendered (outputs undefined, no OOB access)
    reinterpret_cast<uint2*>(ranges)[i] = empty ? make_uint2(0u, 0u) : make_uint2(st, en);
    cursor[(size_t)i * kCtrStride] = st;             // the scatter appends at cursor++ (the sort kernel clears it again)
    len = empty ? 0u : en - st;
  }
  // long lists go to the worklists (warp-aggregated appends): [0, tiles) 4-warp merge kernel, [tiles, 2 tiles) 16-warp merge
  // kernel, [2 tiles, 3 tiles) large kernel; wl_count[0..2] = their lengths
  const int cls = len <= (uint32_t)kTileSortSmallMax ? -1 : (len <= (uint32_t)kTileSortMergeMax ? 0 : (len <= (uint32_t)kTileSortMerge16Max ? 1 : 2));
  const unsigned lt = (1u << lane) - 1u;
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    const unsigned m = __ballot_sync(0xffffffffu, cls == k);
    uint32_t b = 0;
    if (lane == 0 && m) b = atomicAdd(wl_count + k, (uint32_t)__popc(m));
    b = __shfl_sync(0xffffffffu, b, 0);
    if (cls == k) worklist[(size_t)k * tiles + b + __popc(m & lt)] = (uint32_t)i;
  }
}

// Appends (depth bits << 32 | surfel id) to the segment of every tile of the surfel's rect: position = cursor[tile]++ (the
// cursors start at the tiles' first positions).  The returning atomics of up to four tiles are issued back to back
// before the first store (one L2 round trip instead of four).
__global__ void __launch_bounds__(256) tile_scatter_kernel(int N, int TX, const ushort4* __restrict__ rect,
                                                           const uint32_t* __restrict__ count,
                                                           const uint32_t* __restrict__ depth_key, uint32_t* __restrict__ cursor,
                                                           const Status* __restrict__ status, uint64_t* __restrict__ entries) {
  if (status->overflow) return;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int lane = threadIdx.x & 31;
  uint32_t cnt = 0, dk = 0;
  ushort4 r = make_ushort4(0, 0, 0, 0);
  if (i < N) {
    cnt = count[i];
    if (cnt) { dk = depth_key[i]; r = rect[i]; }
  }
  if (cnt && cnt <= kDupCoopThreshold) {
    const uint64_t e = ((uint64_t)dk << 32) | (uint32_t)i;
    const uint32_t w = (uint32_t)(r.z - r.x);
    for (uint32_t q0 = 0; q0 < cnt; q0 += 4) {
      uint32_t pos[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const uint32_t q = q0 + k;
        if (q < cnt) pos[k] = atomicAdd(cursor + (size_t)((r.y + q / w) * TX + r.x + q % w) * kCtrStride, 1u);
      }
#pragma unroll
      for (int k = 0; k < 4; ++k)
        if (q0 + k < cnt) entries[pos[k]] = e;
    }
  }
  unsigned big = __ballot_sync(0xffffffffu, cnt > kDupCoopThreshold);
  while (big) {
    const int src = __ffs(big) - 1;
    big &= big - 1;
    const uint32_t c2 = __shfl_sync(0xffffffffu, cnt, src);
    const uint32_t k2 = __shfl_sync(0xffffffffu, dk, src);
    const int x0 = __shfl_sync(0xffffffffu, (int)r.x, src), y0 = __shfl_sync(0xffffffffu, (int)r.y, src);
    const int x1 = __shfl_sync(0xffffffffu, (int)r.z, src);
    const uint32_t id = (uint32_t)((blockIdx.x * blockDim.x + (threadIdx.x & ~31)) + src);
    const int w = x1 - x0;
    const uint64_t e = ((uint64_t)k2 << 32) | id;
    for (uint32_t q = lane; q < c2; q += 32) {
      const int t = (y0 + (int)(q / (uint32_t)w)) * TX + x0 + (int)(q % (uint32_t)w);
      entries[atomicAdd(cursor + (size_t)t * kCtrStride, 1u)] = e;
    }
  }
}

// Bitonic sort, all comparisons ascending (flip + half-cleaner form), so indices >= n behave as +inf padding and
// are simply skipped.  `buf` may point to shared or global memory; `sync` is __syncwarp or __syncthreads.
template <typename Sync>
__device__ __forceinline__ void bitonic_sort_asc(uint64_t* buf, uint32_t n, uint32_t tid, uint32_t nthreads, Sync sync) {
  uint32_t P = 2;
  while (P < n) P <<= 1;
  for (uint32_t k = 2; k <= P; k <<= 1) {
    {  // flip: a = base + off, b = base + k - 1 - off
      const uint32_t h = k >> 1;
      for (uint32_t i = tid; i < (P >> 1); i += nthreads) {
        const uint32_t base = (i / h) * k, off = i & (h - 1);
        const uint32_t a = base + off, b = base + k - 1 - off;
        if (b < n) {
          const uint64_t x = buf[a], y = buf[b];
          if (x > y) { buf[a] = y; buf[b] = x; }
        }
      }
      sync();
    }
    for (uint32_t j = k >> 2; j > 0; j >>= 1) {
      for (uint32_t i = tid; i < (P >> 1); i += nthreads) {
        const uint32_t a = ((i & ~(j - 1)) << 1) | (i & (j - 1)), b = a + j;
        if (b < n) {
          const uint64_t x = buf[a], y = buf[b];
          if (x > y) { buf[a] = y; buf[b] = x; }
        }
      }
      sync();
    }
  }
}

constexpr int kTileSortWarps = 8;         // warps (= tiles) per CTA
constexpr int kTileSortCtaMax = 16384;    // entries one CTA sorts in shared memory (large-tile kernel)

// Warp-wide bitonic sort of 32*E 64-bit values held in registers, blocked layout: element index of v[e] is
// lane*E + e.  Strides >= E exchange through shuffles (run-time loop: the body is the same for every stride), strides
// below E are register-to-register.  Only the loop over e is unrolled, so the code stays small (an earlier fully
// unrolled version spent 40 % of its issue slots waiting on the instruction cache).
template <int E>
__device__ __forceinline__ void warp_bitonic_regs(uint64_t (&v)[E], int lane) {
  for (int k = 2; k <= 32 * E; k <<= 1) {
    for (int j = k >> 1; j >= E; j >>= 1) {           // partner in another lane (k > j >= E: direction is per lane)
      const int m = j / E;
      const bool take_min = ((lane & m) == 0) == (((lane * E) & k) == 0);
#pragma unroll
      for (int e = 0; e < E; ++e) {
        const uint64_t x = v[e];
        const uint64_t y = __shfl_xor_sync(0xffffffffu, x, m);
        v[e] = ((x < y) == take_min) ? x : y;
      }
    }
#pragma unroll
    for (int js = E >> 1; js >= 1; js >>= 1) {        // partner in this lane's registers
      if (js < k) {
#pragma unroll
        for (int e = 0; e < E; ++e) {
          if ((e & js) == 0) {
            const bool up = (((lane * E + e) & k) == 0);
            const uint64_t x = v[e], y = v[e | js];
            const bool sw = (x > y) == up;
            v[e] = sw ? y : x;
            v[e | js] = sw ? x : y;
          }
        }
      }
    }
  }
}

template <int E>
__device__ __noinline__ void tile_sort_warp(const uint64_t* __restrict__ in, uint32_t n, uint64_t hi, uint64_t* __restrict__ keys,
                                            uint32_t* __restrict__ vals, int lane) {
  uint64_t v[E];
#pragma unroll
  for (int e = 0; e < E; ++e) {
    const uint32_t i = lane * E + e;
    v[e] = i < n ? in[i] : ~0ull;                     // +inf padding sorts to the end (real entries are unique)
  }
  warp_bitonic_regs<E>(v, lane);
#pragma unroll
  for (int e = 0; e < E; ++e) {
    const uint32_t i = lane * E + e;
    if (i < n) {
      keys[i] = hi | (v[e] >> 32);
      vals[i] = (uint32_t)v[e];
    }
  }
}

// same, sorted (depth, id) composites left in shared memory (a chunk of the merge kernel)
template <int E>
__device__ __noinline__ void chunk_sort_warp(const uint64_t* __restrict__ in, uint32_t n, uint64_t* __restrict__ out, int lane) {
  uint64_t v[E];
#pragma unroll
  for (int e = 0; e < E; ++e) {
    const uint32_t i = lane * E + e;
    v[e] = i < n ? in[i] : ~0ull;
  }
  warp_bitonic_regs<E>(v, lane);
#pragma unroll
  for (int e = 0; e < E; ++e) {
    const uint32_t i = lane * E + e;
    if (i < n) out[i] = v[e];
  }
}

// Tiles are dispatched by list length: <= 256 entries here (one warp per tile, 2 / 4 / 8 registers per lane), 257..1024 and
// 1025..4096 in tile_sort_merge_kernel<4> / <16> (one 4- / 16-warp CTA per tile), longer ones in tile_sort_large_kernel
// (one 1024-thread CTA per tile).
// At C3 a fifth of the tiles hold more than 256 entries (walls stack surfels along the ray) and carry half of the
// pairs.  Worklists: [0, tiles) 4-warp merge, [tiles, 2 tiles) 16-warp merge, [2 tiles, 3 tiles) large; wl_count[0..2] = lengths.
__global__ void __launch_bounds__(kTileSortWarps * 32) tile_sort_kernel(int tiles, const uint32_t* __restrict__ ranges,
                                                                        const uint64_t* __restrict__ entries,
                                                                        uint64_t* __restrict__ keys, uint32_t* __restrict__ vals,
                                                                        uint32_t* __restrict__ cursor) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int t = blockIdx.x * kTileSortWarps + warp;
  if (t >= tiles) return;
  if (lane == 0) cursor[(size_t)t * kCtrStride] = 0;   // leave the per-tile counters zero for the next preprocess on this context
  const uint32_t s = ranges[2 * t], n = ranges[2 * t + 1] - s;
  if (n == 0) return;
  if (n > (uint32_t)kTileSortSmallMax) return;   // on a worklist (built by the scan): sorted by the merge / large kernels beside this one
  const uint64_t hi = (uint64_t)(uint32_t)t << 32;
  if (n <= 64) tile_sort_warp<2>(entries + s, n, hi, keys + s, vals + s, lane);
  else if (kTileSortSmallMax <= 128 || n <= 128) tile_sort_warp<4>(entries + s, n, hi, keys + s, vals + s, lane);
  else tile_sort_warp<8>(entries + s, n, hi, keys + s, vals + s, lane);
}

// Lists of 257..4096 entries: the CTA's W warps each sort one W-th in registers (<= 256 entries, 2/4/8 per lane), then
// log2(W) merge rounds in shared memory along merge paths (a thread finds its place on the diagonal by one binary search
// and merges four outputs sequentially; the (depth, id) composites are distinct).
// W = 4 takes the lists up to 1024 entries (C3: a fifth of the tiles), W = 16 those up to 4096 (C1: 200 K surfels on
// 1024 tiles give lists of 1000-2200 entries, which the one-CTA bitonic sort of tile_sort_large_kernel took 60 us for).
template <int W>
__global__ void __launch_bounds__(32 * W) tile_sort_merge_kernel(const uint32_t* __restrict__ ranges, const uint64_t* __restrict__ entries,
                                                                 uint64_t* __restrict__ keys, uint32_t* __restrict__ vals,
                                                                 const uint32_t* __restrict__ worklist, const uint32_t* __restrict__ wl_len) {
  extern __shared__ uint64_t s_merge[];              // two buffers of 256 W composites
  uint64_t* buf_a = s_merge;
  uint64_t* buf_b = s_merge + 256 * W;
  constexpr uint32_t kThreads = 32 * W;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t total = *wl_len;
  // items are dealt round-robin to the CTAs: a shared work counter costs one same-address atomic per item
  for (uint32_t item = blockIdx.x; item < total; item += gridDim.x) {
    __syncthreads();
    const uint32_t t = worklist[item];
    const uint32_t s = ranges[2 * t], n = ranges[2 * t + 1] - s;
    // run length: the smallest of 64 / 128 / 256 that covers the list with W runs, so that the register networks run
    // full (a 350-entry list is three runs of 128 on three warps, not four padded runs of 88)
    const uint32_t c = n <= 64u * W ? 64u : (n <= 128u * W ? 128u : 256u);
    {
      const uint32_t b = min((uint32_t)warp * c, n), e = min(b + c, n), m = e - b;
      if (m > 128u) chunk_sort_warp<8>(entries + s + b, m, buf_a + b, lane);
      else if (m > 64u) chunk_sort_warp<4>(entries + s + b, m, buf_a + b, lane);
      else if (m > 0u) chunk_sort_warp<2>(entries + s + b, m, buf_a + b, lane);
    }
    __syncthreads();
    const uint64_t hi = (uint64_t)t << 32;
    uint64_t* src = buf_a;
    uint64_t* dst = buf_b;
#pragma unroll 1
    for (uint32_t run = c; run < n; run <<= 1) {             // merge pairs of runs of length `run`
      const bool last = (run << 1) >= n;                     // the last round goes straight to the output
      // merge path: a thread produces 4 consecutive outputs; one binary search along the diagonal finds how many of the
      // outputs before them come from the first run, then it merges sequentially (runs start at multiples of 4, so a
      // segment never straddles two pairs)
      for (uint32_t o0 = 4u * threadIdx.x; o0 < n; o0 += 4u * kThreads) {
        const uint32_t pbase = (o0 / (2u * run)) * (2u * run);
        const uint32_t la = min(run, n - pbase), lb = min(run, n - pbase - la);
        const uint64_t* A = src + pbase;
        const uint64_t* B = A + la;
        const uint32_t d = o0 - pbase;
        uint32_t lo = d > lb ? d - lb : 0u, hi_ = min(d, la);
        while (lo < hi_) {
          const uint32_t mid = (lo + hi_) >> 1;
          if (A[mid] < B[d - 1u - mid]) lo = mid + 1u; else hi_ = mid;
        }
        uint32_t i = lo, j = d - lo;
        const uint32_t cnt = min(4u, la + lb - d);
        uint64_t a = i < la ? A[i] : ~0ull, b = j < lb ? B[j] : ~0ull;
#pragma unroll
        for (uint32_t k = 0; k < 4u; ++k) {
          if (k < cnt) {
            const bool ta = a < b;                            // composites are distinct; ~0 marks an exhausted run
            const uint64_t x = ta ? a : b;
            if (ta) { ++i; a = i < la ? A[i] : ~0ull; } else { ++j; b = j < lb ? B[j] : ~0ull; }
            if (last) {
              keys[s + o0 + k] = hi | (x >> 32);
              vals[s + o0 + k] = (uint32_t)x;
            } else {
              dst[o0 + k] = x;
            }
          }
        }
      }
      __syncthreads();
      uint64_t* tmp = src; src = dst; dst = tmp;
    }
  }
}

// tiles with more than kTileSortMergeMax entries (oversized splats; tiny images): one 1024-thread CTA
// per worklist item, in shared memory up to kTileSortCtaMax entries, else in place in global memory.
__global__ void __launch_bounds__(1024) tile_sort_large_kernel(const uint32_t* __restrict__ ranges, uint64_t* __restrict__ entries,
                                                               uint64_t* __restrict__ keys, uint32_t* __restrict__ vals,
                                                               const uint32_t* __restrict__ worklist, uint32_t* __restrict__ wl_count) {
  extern __shared__ uint64_t s_big[];
  const uint32_t total = wl_count[2];   // lists beyond the 16-warp merge kernel
  for (uint32_t item = blockIdx.x; item < total; item += gridDim.x) {
    __syncthreads();
    const uint32_t t = worklist[item];
    const uint32_t s = ranges[2 * t], n = ranges[2 * t + 1] - s;
    uint64_t* buf;
    if (n <= (uint32_t)kTileSortCtaMax) {
      buf = s_big;
      for (uint32_t i = threadIdx.x; i < n; i += 1024) buf[i] = entries[s + i];
    } else {
      buf = entries + s;
    }
    __syncthreads();
    bitonic_sort_asc(buf, n, threadIdx.x, 1024, [] { __syncthreads(); });
    const uint64_t hi = (uint64_t)t << 32;
    for (uint32_t i = threadIdx.x; i < n; i += 1024) {
      const uint64_t v = buf[i];
      keys[s + i] = hi | (v >> 32);
      vals[s + i] = (uint32_t)v;
    }
  }
}

cudaError_t init_binning_attrs() {
  cudaError_t e = cudaFuncSetAttribute(tile_sort_large_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kTileSortCtaMax * 8);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(tile_sort_merge_kernel<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, 2 * 256 * 16 * 8);
  return e;
}

cudaError_t launch_tile_scan(satsplat_ctx* c, cudaStream_t s) {
  const int tiles = c->cam.TX * c->cam.TY;
  const int nblocks = (tiles + kTileScanChunk - 1) / kTileScanChunk;
  g_kernel_launches += 2;
  tile_scan_partial_kernel<<<nblocks, kTileScanThreads, 0, s>>>(tiles, c->tile_count, c->tile_start, c->block_sums, c->wl_count);
  tile_scan_finish_kernel<<<(tiles + kTileScanThreads - 1) / kTileScanThreads, kTileScanThreads, 0, s>>>(tiles, nblocks, c->tile_count, c->tile_start, c->block_sums, c->ranges,
                                                              c->status, (uint32_t)c->max_dup, c->wl_count, c->worklist);
  return cudaGetLastError();
}

cudaError_t launch_tile_scatter(satsplat_ctx* c, int64_t N, cudaStream_t s) {
  if (N == 0) return cudaSuccess;
  ++g_kernel_launches;
  tile_scatter_kernel<<<(int)((N + 255) / 256), 256, 0, s>>>((int)N, c->cam.TX, reinterpret_cast<const ushort4*>(c->rect), c->count,
                                                             c->depth_key, c->tile_count, c->status, c->keys[1]);
  return cudaGetLastError();
}

cudaError_t launch_tile_sort(satsplat_ctx* c, cudaStream_t s) {
  const int tiles = c->cam.TX * c->cam.TY;
  g_kernel_launches += 4;
  // the four kernels work on disjoint tiles (the worklists come from the scan): the long lists are sorted on a second
  // stream beside the many short ones
  // a failed fork would let the side-stream sorts race the scatter on keys[1], a failed join would let the blend read
  // unsorted lists: every event call is checked
  cudaError_t e = cudaEventRecord(c->bin_ev[0], s);
  if (e == cudaSuccess) e = cudaStreamWaitEvent(c->bin_stream, c->bin_ev[0], 0);
  if (e != cudaSuccess) return e;
  tile_sort_merge_kernel<4><<<c->sm_count * 8, 128, 2 * 256 * 4 * 8, c->bin_stream>>>(c->ranges, c->keys[1], c->keys[0], c->vals[0],
                                                                                      c->worklist, c->wl_count + 0);
  tile_sort_merge_kernel<16><<<c->sm_count * 2, 512, 2 * 256 * 16 * 8, c->bin_stream>>>(c->ranges, c->keys[1], c->keys[0], c->vals[0],
                                                                                        c->worklist + tiles, c->wl_count + 1);
  tile_sort_large_kernel<<<(c->sm_count + 1) / 2, 1024, kTileSortCtaMax * 8, c->bin_stream>>>(c->ranges, c->keys[1], c->keys[0], c->vals[0],
                                                                                               c->worklist + 2 * (size_t)tiles, c->wl_count);
  e = cudaEventRecord(c->bin_ev[1], c->bin_stream);
  tile_sort_kernel<<<(tiles + kTileSortWarps - 1) / kTileSortWarps, kTileSortWarps * 32, 0, s>>>(tiles, c->ranges, c->keys[1], c->keys[0],
                                                                                                 c->vals[0], c->tile_count);
  if (e == cudaSuccess) e = cudaStreamWaitEvent(s, c->bin_ev[1], 0);
  if (e != cudaSuccess) {   // no join: do not let the caller's stream run ahead of the side-stream sorts
    cudaStreamSynchronize(c->bin_stream);
    return e;
  }
  c->sorted = 0;
  return cudaGetLastError();
}

}  // namespace satsplat
