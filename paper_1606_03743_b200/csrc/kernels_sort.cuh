// Step a2, first half: spatial binning of the FIELD POINTS.
//
// The adaptive kernel picks one rule per (element, tile of 32R field points) from the tile's
// bounding sphere (the rule follows the distance ratio).  The tighter the
// sphere, the fewer elements fall into a band-straddling shell where the tile has to take the more
// accurate (more expensive) rule, or the pair-by-pair path.  Callers hand field points in any
// order (config 4: along helical tracks, a 128-point tile spans > 2 m), so the points are put in
// Morton (Z-curve) order first: 10 bits per axis over their bounding box, stable LSD radix sort
// of (key, original index), 4 passes of 8 bits.  Everything downstream works on the permuted
// points; reduce_scale_kernel scatters the results back to the caller's order.
//
// The sort is deterministic (stable, no atomics on positions), so tiles - and with them every
// rounding-level detail of the result - are reproducible from run to run.
#pragma once
#include "device_utils.cuh"

namespace bemcub {

constexpr int kSortChunk = 1024;  // keys per warp-sized block in the radix passes
constexpr int kRadixBits = 8;
constexpr int kRadix = 1 << kRadixBits;

// order-preserving map double -> uint64 (for atomicMin / atomicMax on coordinates)
__device__ __forceinline__ unsigned long long ordered_bits(double x) {
  const unsigned long long b = (unsigned long long)__double_as_longlong(x);
  return (b >> 63) ? ~b : (b | 0x8000000000000000ull);
}
__device__ __forceinline__ double from_ordered_bits(unsigned long long u) {
  const unsigned long long b = (u >> 63) ? (u & 0x7fffffffffffffffull) : ~u;
  return __longlong_as_double((long long)b);
}

// box[0..2] = min x,y,z ; box[3..5] = max x,y,z (ordered bits; mins preset to ~0, maxs to 0).
// Non-finite coordinates are ignored here and clamped into the box by morton_key_kernel.
__global__ void bbox_kernel(int64_t m, const double* __restrict__ pts, unsigned long long* __restrict__ box) {
  double lo[3] = {CUDART_INF, CUDART_INF, CUDART_INF}, hi[3] = {-CUDART_INF, -CUDART_INF, -CUDART_INF};
  for (int64_t j = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; j < m; j += (int64_t)gridDim.x * blockDim.x) {
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      const double v = pts[3 * j + a];
      if (isfinite(v)) {
        lo[a] = fmin(lo[a], v);
        hi[a] = fmax(hi[a], v);
      }
    }
  }
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    lo[a] = warp_min(lo[a]);
    hi[a] = warp_max(hi[a]);
  }
  if ((threadIdx.x & 31) == 0) {
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      if (lo[a] <= hi[a]) {
        atomicMin(box + a, ordered_bits(lo[a]));
        atomicMax(box + 3 + a, ordered_bits(hi[a]));
      }
    }
  }
}

__device__ __forceinline__ uint32_t spread10(uint32_t v) {  // 10 bits -> every third bit
  v &= 0x3ffu;
  v = (v | (v << 16)) & 0x030000ffu;
  v = (v | (v << 8)) & 0x0300f00fu;
  v = (v | (v << 4)) & 0x030c30c3u;
  v = (v | (v << 2)) & 0x09249249u;
  return v;
}

__global__ void morton_key_kernel(int64_t m, const double* __restrict__ pts, const unsigned long long* __restrict__ box,
                                  uint32_t* __restrict__ key, uint32_t* __restrict__ idx) {
  const int64_t j = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (j >= m) return;
  uint32_t q[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    const double lo = from_ordered_bits(box[a]), hi = from_ordered_bits(box[3 + a]);
    const double ext = hi - lo;
    const double s = (ext > 0.0 && isfinite(ext)) ? 1024.0 / ext : 0.0;
    const double t = (pts[3 * j + a] - lo) * s;
    q[a] = (uint32_t)fmin(fmax(t, 0.0), 1023.0);  // NaN -> 0
  }
  key[j] = spread10(q[0]) | (spread10(q[1]) << 1) | (spread10(q[2]) << 2);
  idx[j] = (uint32_t)j;
}

// ---- stable LSD radix sort, one warp per chunk of kSortChunk keys -------------------------------
// pass 1: hist[d * nblocks + b] = number of keys of chunk b whose digit is d
__global__ void __launch_bounds__(32) radix_hist_kernel(int64_t m, const uint32_t* __restrict__ key, int shift, int nblocks,
                                                        uint32_t* __restrict__ hist) {
  __shared__ uint32_t cnt[kRadix];
  const int lane = threadIdx.x;
  for (int d = lane; d < kRadix; d += 32) cnt[d] = 0;
  __syncwarp();
  const int64_t base = (int64_t)blockIdx.x * kSortChunk;
  for (int i = lane; i < kSortChunk; i += 32) {
    const int64_t j = base + i;
    if (j < m) atomicAdd(&cnt[(key[j] >> shift) & (kRadix - 1)], 1u);
  }
  __syncwarp();
  for (int d = lane; d < kRadix; d += 32) hist[(size_t)d * nblocks + blockIdx.x] = cnt[d];
}

// pass 2: exclusive scan of the digit-major histogram (one block; `total` entries)
__global__ void __launch_bounds__(1024) radix_scan_kernel(int64_t total, uint32_t* __restrict__ hist) {
  __shared__ uint32_t wsum[32];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int64_t per = (total + 1023) / 1024;
  const int64_t lo = tid * per, hi = min(total, lo + per);
  uint32_t s = 0;
  for (int64_t i = lo; i < hi; ++i) s += hist[i];
  // block-wide exclusive scan of the per-thread sums
  uint32_t x = s;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const uint32_t y = __shfl_up_sync(kFullMask, x, o);
    if (lane >= o) x += y;
  }
  if (lane == 31) wsum[warp] = x;
  __syncthreads();
  if (warp == 0) {
    uint32_t w = wsum[lane];
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t y = __shfl_up_sync(kFullMask, w, o);
      if (lane >= o) w += y;
    }
    wsum[lane] = w;
  }
  __syncthreads();
  uint32_t run = (x - s) + (warp > 0 ? wsum[warp - 1] : 0u);
  for (int64_t i = lo; i < hi; ++i) {
    const uint32_t v = hist[i];
    hist[i] = run;
    run += v;
  }
}

// pass 3: stable scatter.  Keys of a chunk are visited 32 at a time in index order; equal digits
// inside a group are ranked by lane (match_any), groups are sequential, so ties keep their order.
__global__ void __launch_bounds__(32) radix_scatter_kernel(int64_t m, const uint32_t* __restrict__ key_in,
                                                           const uint32_t* __restrict__ idx_in, int shift, int nblocks,
                                                           const uint32_t* __restrict__ hist, uint32_t* __restrict__ key_out,
                                                           uint32_t* __restrict__ idx_out) {
  __shared__ uint32_t pos[kRadix];
  const int lane = threadIdx.x;
  for (int d = lane; d < kRadix; d += 32) pos[d] = hist[(size_t)d * nblocks + blockIdx.x];
  __syncwarp();
  const int64_t base = (int64_t)blockIdx.x * kSortChunk;
  for (int i = 0; i < kSortChunk; i += 32) {
    const int64_t j = base + i + lane;
    const bool ok = j < m;
    if (!__any_sync(kFullMask, ok)) break;
    const uint32_t k = ok ? key_in[j] : 0u;
    const uint32_t v = ok ? idx_in[j] : 0u;
    const uint32_t d = ok ? ((k >> shift) & (kRadix - 1)) : (uint32_t)kRadix;  // sentinel groups the idle lanes
    const unsigned peers = __match_any_sync(kFullMask, d);
    const int rank = __popc(peers & ((1u << lane) - 1u));
    const int leader = __ffs(peers) - 1;
    uint32_t start = 0;
    if (ok && lane == leader) start = pos[d];
    start = __shfl_sync(kFullMask, start, leader);
    __syncwarp();
    if (ok && lane == leader) pos[d] = start + (uint32_t)__popc(peers);
    __syncwarp();
    if (ok) {
      key_out[start + rank] = k;
      idx_out[start + rank] = v;
    }
  }
}

// sorted[j] = pts[idx[j]]
__global__ void gather_points_kernel(int64_t m, const double* __restrict__ pts, const uint32_t* __restrict__ idx,
                                     double* __restrict__ sorted) {
  const int64_t j = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (j >= m) return;
  const int64_t s = idx[j];
  sorted[3 * j] = pts[3 * s];
  sorted[3 * j + 1] = pts[3 * s + 1];
  sorted[3 * j + 2] = pts[3 * s + 2];
}

}  // namespace bemcub
