// matrix-free solve of the BEM collocation system
//     sum_j A_ij sigma_j = V_i,   A_ij = k Int_{element j} dS / |c_i - Q|,
// for the unknown charge densities, without ever storing A ("shell matrices", L200): the mat-vec
// is the potential-only adaptive evaluation kernel at the element centroids (analytic self and
// near terms by the distance-ratio policy, L159).  This file holds the small vector kernels of
// the restarted GMRES iteration around it; all reductions are deterministic (fixed tree, no
// atomics), so a solve is reproducible bit for bit.
#pragma once
#include "analytic.cuh"
#include "device_utils.cuh"

namespace bemcub {

// diag[i] = A_ii = k * (analytic potential integral of element i at its own centroid); the right
// (Jacobi) preconditioner of the iteration.
__global__ void self_term_kernel(int64_t n, const uint8_t* __restrict__ type, const double* __restrict__ verts,
                                 const double4* __restrict__ cenL, double k, double* __restrict__ diag) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= n) return;
  Vec3 V[4];
  const int nv = load_polygon(type, verts, i, V);
  const double4 c = cenL[i];
  double ip;
  Vec3 ie;
  analytic_integrals<false>(V, nv, Vec3{c.x, c.y, c.z}, ip, ie);
  diag[i] = k * ip;
}

// out[v] = V[v] . w for v < nvec (one block per vector; V[v] = basis + v * ld)
__global__ void __launch_bounds__(1024) vec_dots_kernel(int64_t n, const double* __restrict__ basis, int64_t ld,
                                                        const double* __restrict__ w, double* __restrict__ out) {
  __shared__ double red[32];
  const double* v = basis + (int64_t)blockIdx.x * ld;
  double s = 0.0;
  for (int64_t i = threadIdx.x; i < n; i += blockDim.x) s = fma(v[i], w[i], s);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(kFullMask, s, o);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
  __syncthreads();
  if (threadIdx.x < 32) {
    s = threadIdx.x < (blockDim.x >> 5) ? red[threadIdx.x] : 0.0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(kFullMask, s, o);
    if (threadIdx.x == 0) out[blockIdx.x] = s;
  }
}

// w += sign * sum_{v < nvec} coef[v] * V[v]      (coef in device memory)
__global__ void vec_combine_kernel(int64_t n, int nvec, const double* __restrict__ basis, int64_t ld,
                                   const double* __restrict__ coef, double sign, double* __restrict__ w) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= n) return;
  double s = 0.0;
  for (int v = 0; v < nvec; ++v) s = fma(coef[v], basis[(int64_t)v * ld + i], s);
  w[i] = fma(sign, s, w[i]);
}

// dst = alpha * a / (d ? d : 1)          (scaling of a basis vector; preconditioner application)
__global__ void vec_scale_kernel(int64_t n, double alpha, const double* __restrict__ a, const double* __restrict__ d,
                                 double* __restrict__ dst) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= n) return;
  dst[i] = d ? alpha * a[i] / d[i] : alpha * a[i];
}

// dst = a - b   (dst may be b: no __restrict__ on those two)
__global__ void vec_sub_kernel(int64_t n, const double* __restrict__ a, const double* b, double* dst) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i < n) dst[i] = a[i] - b[i];
}

// dst = a / sqrt(*norm2)   (normalisation by a squared norm that is still on the device; 0 -> copy)
__global__ void vec_normalise_kernel(int64_t n, const double* __restrict__ a, const double* __restrict__ norm2, double* __restrict__ dst) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= n) return;
  const double s = *norm2;
  dst[i] = s > 0.0 ? a[i] / sqrt(s) : a[i];
}

// x += u / d
__global__ void vec_add_scaled_kernel(int64_t n, const double* __restrict__ u, const double* __restrict__ d, double* __restrict__ x) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i < n) x[i] += u[i] / d[i];
}

// out[i] = sum_j A[i * ld + j] x[j]: the mat-vec of a solve whose matrix is kept in device memory
// (bemcub_solve_storage).  Bound by the HBM read of the 8 n^2 bytes of A: one CTA takes one row at a
// time, every thread 16-byte streaming loads, four in flight; x comes from L1 / L2.  The sums are
// combined in a fixed order (four per thread, warp shuffles, the warps in index order).
constexpr int kGemvThreads = 256;
constexpr int kGemvCtasPerSm = 8;
__global__ void __launch_bounds__(kGemvThreads) gemv_rows_kernel(int64_t n, const double* __restrict__ A, int64_t ld,
                                                                 const double* __restrict__ x, double* __restrict__ out) {
  __shared__ double red[kGemvThreads / 32];
  constexpr int T = kGemvThreads;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const bool vec = ((ld & 1) == 0) && ((reinterpret_cast<uintptr_t>(A) & 15u) == 0) && ((reinterpret_cast<uintptr_t>(x) & 15u) == 0);
  for (int64_t i = blockIdx.x; i < n; i += gridDim.x) {
    const double* row = A + i * ld;
    double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
    if (vec) {
      const double2* r2 = reinterpret_cast<const double2*>(row);
      const double2* x2 = reinterpret_cast<const double2*>(x);
      const int64_t n2 = n >> 1;
      int64_t j = threadIdx.x;
      for (; j + 3 * T < n2; j += 4 * T) {
        const double2 a0 = __ldcs(r2 + j), a1 = __ldcs(r2 + j + T), a2 = __ldcs(r2 + j + 2 * T), a3 = __ldcs(r2 + j + 3 * T);
        const double2 b0 = x2[j], b1 = x2[j + T], b2 = x2[j + 2 * T], b3 = x2[j + 3 * T];
        s0 = fma(a0.y, b0.y, fma(a0.x, b0.x, s0));
        s1 = fma(a1.y, b1.y, fma(a1.x, b1.x, s1));
        s2 = fma(a2.y, b2.y, fma(a2.x, b2.x, s2));
        s3 = fma(a3.y, b3.y, fma(a3.x, b3.x, s3));
      }
      for (; j < n2; j += T) {
        const double2 a0 = __ldcs(r2 + j), b0 = x2[j];
        s0 = fma(a0.y, b0.y, fma(a0.x, b0.x, s0));
      }
      if ((n & 1) && threadIdx.x == 0) s1 = fma(row[n - 1], x[n - 1], s1);
    } else {
      for (int64_t j = threadIdx.x; j < n; j += T) s0 = fma(__ldcs(row + j), x[j], s0);
    }
    double s = (s0 + s1) + (s2 + s3);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(kFullMask, s, o);
    if (lane == 0) red[warp] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
      double t = 0.0;
#pragma unroll
      for (int w = 0; w < T / 32; ++w) t += red[w];
      out[i] = t;
    }
    __syncthreads();
  }
}

}  // namespace bemcub
