// Step a1 of the hot path: element preprocessing.
//   geometry_kernel : per element centroid Q_cen, area A, mean side L, validity
//   expand_kernel   : per (element, rule point) the Gaussian point Q_i by Eq. 3.3 (triangle, L109)
//                     or Eq. 3.2 (rectangle, L103) and its charge q_i = w_i sigma A (L143),
//                     stored as one packed (x,y,z,q) record per point, one array per rule level.
#pragma once
#include "device_utils.cuh"

namespace bemcub {

// Rule tables in constant memory, filled by bemcub_create from rules.h.
// Triangle: (lambda_A, lambda_B, lambda_C, w) per point; rectangle: (x, y, w, 0).
__constant__ double c_tri_tab[75 * 4];
__constant__ double c_rect_tab[73 * 4];
__constant__ int c_tri_off[6];
__constant__ int c_rect_off[6];

struct GeomStatus {
  int code;  // min over elements of the (negative) error code, 0 = fine
  int pad;
  unsigned long long n_tri, n_rect;
};

// Centroid, mean side L (in c.w) and area of one element from its nine stored coordinates; returns
// 0 or the (negative) error code of include/bemcub.h.
__device__ __forceinline__ int element_geometry(int t, const double* __restrict__ v, double4& c, double& A) {
  const double ax = v[0], ay = v[1], az = v[2];
  const double e1x = v[3] - ax, e1y = v[4] - ay, e1z = v[5] - az;
  const double e2x = v[6] - ax, e2y = v[7] - ay, e2z = v[8] - az;
  int code = 0;
  if (t == 0) {
    // triangle A,B,C: area = |AB x AC|/2, centroid = (A+B+C)/3, L = (|AB|+|BC|+|CA|)/3
    const double nx = e1y * e2z - e1z * e2y, ny = e1z * e2x - e1x * e2z, nz = e1x * e2y - e1y * e2x;
    A = 0.5 * sqrt(nx * nx + ny * ny + nz * nz);
    c.x = (ax + v[3] + v[6]) / 3.0;
    c.y = (ay + v[4] + v[7]) / 3.0;
    c.z = (az + v[5] + v[8]) / 3.0;
    const double bx = v[6] - v[3], by = v[7] - v[4], bz = v[8] - v[5];
    c.w = (sqrt(e1x * e1x + e1y * e1y + e1z * e1z) + sqrt(bx * bx + by * by + bz * bz) +
           sqrt(e2x * e2x + e2y * e2y + e2z * e2z)) / 3.0;
    if (!(A > 0.0)) code = -2;
  } else if (t == 1) {
    // rectangle P0, P1 = P0 + a u_x, P3 = P0 + b u_y: A = ab, centre = P0 + e1/2 + e2/2, L = (a+b)/2
    const double a = sqrt(e1x * e1x + e1y * e1y + e1z * e1z), b = sqrt(e2x * e2x + e2y * e2y + e2z * e2z);
    A = a * b;
    c.x = ax + 0.5 * e1x + 0.5 * e2x;
    c.y = ay + 0.5 * e1y + 0.5 * e2y;
    c.z = az + 0.5 * e1z + 0.5 * e2z;
    c.w = 0.5 * (a + b);
    if (!(a > 0.0) || !(b > 0.0)) code = -2;
    else if (fabs(e1x * e2x + e1y * e2y + e1z * e2z) > 1e-12 * a * b) code = -3;
  } else {
    A = 0.0;
    c = make_double4(0, 0, 0, 0);
    code = -1;
  }
  return code;
}

// cenL[e] = (Q_cen.x, Q_cen.y, Q_cen.z, L); area[e] = A.
__global__ void geometry_kernel(int64_t n, const uint8_t* __restrict__ type, const double* __restrict__ verts,
                                double4* __restrict__ cenL, double* __restrict__ area, GeomStatus* status) {
  const int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (e >= n) return;
  const int t = type[e];
  double4 c;
  double A;
  const int code = element_geometry(t, verts + 9 * e, c, A);
  cenL[e] = c;
  area[e] = A;
  if (code) atomicMin(&status->code, code);
  // element-type census, one atomic per warp
  const unsigned act = __activemask();
  const unsigned tris = __ballot_sync(act, t == 0), rects = __ballot_sync(act, t == 1);
  if ((threadIdx.x & 31) == __ffs(act) - 1) {
    if (tris) atomicAdd(&status->n_tri, (unsigned long long)__popc(tris));
    if (rects) atomicAdd(&status->n_rect, (unsigned long long)__popc(rects));
  }
}

__device__ __forceinline__ int rule_npts_of(int type, int level) {
  return type == 0 ? (c_tri_off[level + 1] - c_tri_off[level]) : (c_rect_off[level + 1] - c_rect_off[level]);
}

// Point i of rule `level` on one element: Q_i by Eq. 3.3 (triangle, L109) or Eq. 3.2 (rectangle,
// L103) and q_i = w_i q sigma(Q_i)/sigma  (q = sigma A; sv != nullptr: linear density, L275).
// The ONE place this arithmetic lives: the preprocessing kernel and the on-the-fly kernel call it,
// so precomputed and on-the-fly points are bit-identical (L218 vs L246).
__device__ __forceinline__ bool rule_point(int t, int level, int i, const double* __restrict__ v, const double4 c, double q,
                                           const double* __restrict__ sv, double4& out) {
  if (t == 0) {
    const double* r = c_tri_tab + 4 * (c_tri_off[level] + i);
    const double la = r[0], lb = r[1], lc = r[2];
    // Eq. 3.3: Q = lambda_A A + lambda_B B + lambda_C C
    out.x = fma(lc, v[6], fma(lb, v[3], la * v[0]));
    out.y = fma(lc, v[7], fma(lb, v[4], la * v[1]));
    out.z = fma(lc, v[8], fma(lb, v[5], la * v[2]));
    const double sq = sv ? fma(lc, sv[2], fma(lb, sv[1], la * sv[0])) : 1.0;
    out.w = r[3] * q * sq;
  } else {
    const double* r = c_rect_tab + 4 * (c_rect_off[level] + i);
    const double xs = 0.5 * r[0], ys = 0.5 * r[1];
    // Eq. 3.2: Q = Q_cen + (a/2) x u_x + (b/2) y u_y, with a u_x = P1 - P0 and b u_y = P3 - P0
    out.x = fma(ys, v[6] - v[0], fma(xs, v[3] - v[0], c.x));
    out.y = fma(ys, v[7] - v[1], fma(xs, v[4] - v[1], c.y));
    out.z = fma(ys, v[8] - v[2], fma(xs, v[5] - v[2], c.z));
    const double sq = sv ? fma(0.5 + ys, sv[2] - sv[0], fma(0.5 + xs, sv[1] - sv[0], sv[0])) : 1.0;
    out.w = r[2] * q * sq;
  }
  return true;
}

// The same point with element type, level and index known at compile time (fully unrolled callers): the
// table entries become constant-bank operands of the FP64 instructions, with no address arithmetic and no
// load instruction - what the kernel for few field points spends most of its non-FP64 instructions on
// otherwise.  Same operations in the same order as rule_point(): bit-identical points.
constexpr int kTriOffCt[6] = {0, 4, 11, 23, 42, 75};   // = c_tri_off / c_rect_off (checked by bemcub_create)
constexpr int kRectOffCt[6] = {0, 4, 11, 23, 40, 73};
template <int T, int LEVEL>
__device__ __forceinline__ void rule_point_ct(int i, const double* __restrict__ v, const double4 c, double q,
                                              const double* __restrict__ sv, double4& out) {
  if constexpr (T == 0) {
    const double* r = c_tri_tab + 4 * (kTriOffCt[LEVEL] + i);
    const double la = r[0], lb = r[1], lc = r[2];
    out.x = fma(lc, v[6], fma(lb, v[3], la * v[0]));
    out.y = fma(lc, v[7], fma(lb, v[4], la * v[1]));
    out.z = fma(lc, v[8], fma(lb, v[5], la * v[2]));
    const double sq = sv ? fma(lc, sv[2], fma(lb, sv[1], la * sv[0])) : 1.0;
    out.w = r[3] * q * sq;
  } else {
    const double* r = c_rect_tab + 4 * (kRectOffCt[LEVEL] + i);
    const double xs = 0.5 * r[0], ys = 0.5 * r[1];
    out.x = fma(ys, v[6] - v[0], fma(xs, v[3] - v[0], c.x));
    out.y = fma(ys, v[7] - v[1], fma(xs, v[4] - v[1], c.y));
    out.z = fma(ys, v[8] - v[2], fma(xs, v[5] - v[2], c.z));
    const double sq = sv ? fma(0.5 + ys, sv[2] - sv[0], fma(0.5 + xs, sv[1] - sv[0], sv[0])) : 1.0;
    out.w = r[2] * q * sq;
  }
}

template <typename T> struct Point4;
template <> struct Point4<double> { typedef double4 type; };
template <> struct Point4<float> { typedef float4 type; };

__device__ __forceinline__ void store_point(double4* dst, double x, double y, double z, double q) {
  *dst = make_double4(x, y, z, q);
}
__device__ __forceinline__ void store_point(float4* dst, double x, double y, double z, double q) {
  *dst = make_float4((float)x, (float)y, (float)z, (float)q);
}

// One thread per (element, slot); slot < stride.  Slots beyond the element's own N are padding:
// zero charge at the position of the element's FIRST Gaussian point (a zero charge adds exactly
// nothing wherever a real charge of the same place gives a finite term; the centroid would not do:
// it is a field point of the matrix fill).  sigma == nullptr means unit sigma (matrix assembly, L34).
// sigma_v != nullptr: the density varies linearly over the element (L275), sigma_v[e][3] = its
// values at the three stored vertices, q_i = w_i A sigma(Q_i) with sigma(Q_i) from the rule's
// reference coordinates (triangle: sum lambda_v sigma_v; rectangle: corner value + the two slopes).
template <typename T>
__global__ void expand_kernel(int64_t n, int level, int stride, const uint8_t* __restrict__ type,
                              const double* __restrict__ verts, const double4* __restrict__ cenL,
                              const double* __restrict__ area, const double* __restrict__ sigma,
                              const double* __restrict__ sigma_v, double scale, typename Point4<T>::type* __restrict__ out) {
  const int64_t idx = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (idx >= n * stride) return;
  const int64_t e = idx / stride;
  const int i = (int)(idx - e * stride);
  const int t = type[e];
  const double* v = verts + 9 * e;
  // q = sigma A (L143); with sigma_v: q = A.  scale = 1 except for the matrix fill, which folds k in.
  const double q = (sigma ? sigma[e] : 1.0) * area[e] * scale;
  const double* sv = sigma_v ? sigma_v + 3 * e : nullptr;
  const double4 c = cenL[e];
  double4 pt;
  const bool real = i < rule_npts_of(t, level);
  rule_point(t, level, real ? i : 0, v, c, q, sv, pt);
  store_point(out + idx, pt.x, pt.y, pt.z, real ? pt.w : 0.0);
}

// Step a6: sum the per-split partial results in split order and apply k = 1/(4 pi eps0) once
// (Eq. 4.1 prefactor, L141).  `perm` (may be null) maps the evaluation order back to the caller's
// field-point order (kernels_sort.cuh).
__global__ void reduce_scale_kernel(int64_t m, int nsplit, int64_t split_stride, const double4* __restrict__ partial,
                                    const double* __restrict__ partial_g, double k, const uint32_t* __restrict__ perm,
                                    double* __restrict__ phi, double* __restrict__ E, double* __restrict__ G) {
  int64_t j = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (j >= m) return;
  // summed in split order; eight loads in flight per thread (a call with few field points and many
  // splits spends its time here waiting for L2 otherwise)
  double4 s = partial[j];
  int sp = 1;
  for (; sp + 8 <= nsplit; sp += 8) {
    double4 p[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) p[u] = partial[(int64_t)(sp + u) * split_stride + j];
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      s.x += p[u].x;
      s.y += p[u].y;
      s.z += p[u].z;
      s.w += p[u].w;
    }
  }
  for (; sp < nsplit; ++sp) {
    const double4 p = partial[(int64_t)sp * split_stride + j];
    s.x += p.x;
    s.y += p.y;
    s.z += p.z;
    s.w += p.w;
  }
  double g[6] = {0, 0, 0, 0, 0, 0};
  if (G) {
    for (int sp = 0; sp < nsplit; ++sp)
#pragma unroll
      for (int c = 0; c < 6; ++c) g[c] += partial_g[(sp * split_stride + j) * 6 + c];
  }
  if (perm) j = perm[j];
  if (phi) phi[j] = k * s.x;
  if (E) {
    E[3 * j] = k * s.y;
    E[3 * j + 1] = k * s.z;
    E[3 * j + 2] = k * s.w;
  }
  if (G) {  // G_ab = k (delta_ab sg - s_ab); traceless: G_zz = -(G_xx + G_yy)
    const double gxx = k * (g[0] - g[1]), gyy = k * (g[0] - g[2]);
    G[6 * j] = gxx;
    G[6 * j + 1] = gyy;
    G[6 * j + 2] = -(gxx + gyy);
    G[6 * j + 3] = -k * g[3];
    G[6 * j + 4] = -k * g[4];
    G[6 * j + 5] = -k * g[5];
  }
}

// Roofline denominator (bemcub_fp64_issue_sweep): 16 (18 for the mix) independent chains per thread of
// one FP64 instruction kind, the second operand in a uniform register so that an instruction reads at
// most two vector registers - the form in which the pipe issues one warp instruction per two cycles
// per scheduler.  MIX 0: DFMA, 1: DADD, 2: DMUL, 3: the 8 DFMA : 6 DMUL : 4 DADD mix of Eq. 4.1.
// Two more mixes are not candidates for the peak but evidence for the issue model the kernels are
// written for: MIX 4: DFMA whose three sources are three different, changing
// vector registers (3 dispatch cycles instead of 2); MIX 5: the DFMA loop of MIX 0 with one integer
// multiply-add after every second DFMA (a non-FP64 instruction takes a dispatch cycle of its own).
// clk[0] = SM cycles, clk[1] = nanoseconds of the launch as thread 0 of CTA 0 saw them.
template <int MIX>
__global__ void fp64_issue_kernel(double* out, unsigned long long* clk, int iters, double a, double b, int ia) {
  constexpr int C = (MIX == 3) ? 18 : 16;
  double x[C];
  int n[8];
#pragma unroll
  for (int k = 0; k < C; ++k) x[k] = 1.0 + (double)(threadIdx.x + k) * 1e-3;
#pragma unroll
  for (int k = 0; k < 8; ++k) n[k] = threadIdx.x + k;
  KernelClock kc;
  kc.begin();
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 4; ++u) {
#pragma unroll
      for (int k = 0; k < C; ++k) {
        if (MIX == 4) x[k] = __fma_rn(x[k], x[(k + 5) % C], x[(k + 11) % C]);
        else if (MIX == 0 || MIX == 5 || (MIX == 3 && k < 8)) x[k] = __fma_rn(x[k], a, b);
        else if (MIX == 1 || (MIX == 3 && k >= 14)) x[k] = __dadd_rn(x[k], b);
        else x[k] = __dmul_rn(x[k], a);
        if (MIX == 5 && (k & 1)) n[k >> 1] = n[k >> 1] * ia + i;
      }
    }
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    clk[0] = (unsigned long long)(clock64() - kc.c0);
    clk[1] = global_timer_ns() - kc.t0;
  }
  double s = 0.0;
#pragma unroll
  for (int k = 0; k < C; ++k) s += x[k];
  if (MIX == 5) {
#pragma unroll
    for (int k = 0; k < 8; ++k) s += (double)n[k];
  }
  out[blockIdx.x * (int64_t)blockDim.x + threadIdx.x] = s;
}

// Resident synthetic data of bemcub_inner_loop_rate: field points 3..4 m away from source points
// in the unit cube (values only need to be finite and distinct).
__global__ void fill_synthetic_kernel(int64_t nfield, double* __restrict__ field, int nsrc, double4* __restrict__ src) {
  const int64_t j = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (j < nfield) {
    field[3 * j] = 3.0 + 1e-4 * (double)(j % 9973);
    field[3 * j + 1] = 2.0 + 1e-4 * (double)(j % 7919);
    field[3 * j + 2] = 1.0 + 1e-4 * (double)(j % 6007);
  }
  if (j < nsrc) src[j] = make_double4(0.001 * (double)j, 0.5 - 0.0007 * (double)j, 0.3 + 0.0003 * (double)j, 1e-9 * (double)(1 + j % 7));
}

}  // namespace bemcub
