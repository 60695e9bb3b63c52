// The single-element boundary integrator (PAPER.md L193-196 item a): element k seen from field point
// k, k < K, no sum over elements - the unit of the paper's accuracy protocol (L68, L149: random
// elements and field-point directions per distance ratio; Figs. 8-10) and of the Duffy comparison
// (L163-169).  One thread per pair: geometry (L66), the rule's points on the fly (Eq. 3.2 / 3.3, the
// same rule_point() as the preprocessing kernel), Eq. 4.1, or the closed form of step a4.
#pragma once
#include "analytic.cuh"
#include "kernels_eval.cuh"
#include "kernels_pre.cuh"

namespace bemcub {

constexpr int kMethodAnalytic = 5, kMethodDuffy0 = 8;

struct PairsParams {
  int64_t K;
  const uint8_t* type;
  const double* verts;
  const double* sigma;  // may be null: unit density
  int method;           // 0..4 rule level, 5 analytic, -1 by distance ratio, 8 + l Duffy-mapped rectangle rule l
  PolicyDev pol;
  const double* field;
  double* phi;
  double* E;  // may be null
  double k;
};

// Point i of the rectangle rule of `level` on a TRIANGLE through the Duffy map (L163-169; DESIGN.md
// reading 20): Q = A + u [(B - A) + v (C - B)], u = (1 + y)/2, v = (1 + x)/2, dS = 2 area u du dv, so
// the weight relative to the area is (1 + y) w.
__device__ __forceinline__ void duffy_point(int level, int i, const double* __restrict__ v, double q, double4& out) {
  const double* r = c_rect_tab + 4 * (c_rect_off[level] + i);
  const double u = 0.5 * (1.0 + r[1]), w = 0.5 * (1.0 + r[0]);
  out.x = fma(u, fma(w, v[6] - v[3], v[3] - v[0]), v[0]);
  out.y = fma(u, fma(w, v[7] - v[4], v[4] - v[1]), v[1]);
  out.z = fma(u, fma(w, v[8] - v[5], v[5] - v[2]), v[2]);
  out.w = (1.0 + r[1]) * r[2] * q;
}

template <typename T>
__global__ void __launch_bounds__(128) eval_pairs_kernel(const __grid_constant__ PairsParams p) {
  const int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (e >= p.K) return;
  const int t = p.type[e];
  double v[9];
#pragma unroll
  for (int k = 0; k < 9; ++k) v[k] = p.verts[9 * e + k];
  double4 c;
  double A;
  const int code = element_geometry(t, v, c, A);
  const double Px = p.field[3 * e], Py = p.field[3 * e + 1], Pz = p.field[3 * e + 2];
  const double sg = p.sigma ? p.sigma[e] : 1.0;
  double phi = 0.0, ex = 0.0, ey = 0.0, ez = 0.0;
  int method = p.method;
  if (method == -1) {
    const double dx = __dsub_rn(Px, c.x), dy = __dsub_rn(Py, c.y), dz = __dsub_rn(Pz, c.z);
    const double D2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
    method = p.pol.map[want_level(D2, c.w, p.pol.dr[t & 1])];
  }
  if (code != 0) {
    phi = ex = ey = ez = CUDART_NAN;  // no integral over a degenerate element
  } else if (method == kMethodAnalytic) {
    Vec3 V[4];
    V[0] = {v[0], v[1], v[2]};
    V[1] = {v[3], v[4], v[5]};
    V[3] = {v[6], v[7], v[8]};
    V[2] = (t == 0) ? V[3] : Vec3{V[1].x + (V[3].x - V[0].x), V[1].y + (V[3].y - V[0].y), V[1].z + (V[3].z - V[0].z)};
    double ip;
    Vec3 ie;
    analytic_integrals<true>(V, t == 0 ? 3 : 4, Vec3{Px, Py, Pz}, ip, ie);
    phi = sg * ip;
    ex = sg * ie.x; ey = sg * ie.y; ez = sg * ie.z;
  } else {
    const bool duffy = method >= kMethodDuffy0 && t == 0;
    const int level = method >= kMethodDuffy0 ? method - kMethodDuffy0 : method;
    const int N = duffy ? rule_npts(1, level) : rule_npts(t, level);
    const double q = sg * A;
    const double c375 = c_three_eighths;
    T fphi = 0, fx = 0, fy = 0, fz = 0;
    for (int i = 0; i < N; ++i) {
      double4 s;
      if (duffy) duffy_point(level, i, v, q, s);
      else rule_point(t, level, i, v, c, q, nullptr, s);
      interact_one((T)s.x, (T)s.y, (T)s.z, (T)s.w, (T)Px, (T)Py, (T)Pz, fphi, fx, fy, fz, c375);
    }
    phi = (double)fphi; ex = (double)fx; ey = (double)fy; ez = (double)fz;
  }
  p.phi[e] = p.k * phi;
  if (p.E) {
    p.E[3 * e] = p.k * ex;
    p.E[3 * e + 1] = p.k * ey;
    p.E[3 * e + 2] = p.k * ez;
  }
}

}  // namespace bemcub
