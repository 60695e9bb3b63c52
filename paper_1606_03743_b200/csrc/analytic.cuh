// Step a4 of the hot path: exact near-field integrals of Eq. 2.1 over a flat
// triangle or rectangle,
//     I_phi = Int dS / |P-Q|,      I_E = Int dS (P-Q) / |P-Q|^3            (unit sigma, no k),
// used below the first distance-ratio limit (L159).  The paper only cites its analytic formulas
// (L68, L78); reading 9 fixes the closed form used here — the classical edge-by-edge
// line-integral form.  For a polygon with unit normal n, height h = n.(P - V0) and, per edge
// V- -> V+ with unit vector l and in-plane outward normal u = l x n:
//     s+- = (V+- - P).l,  t0 = (V- - P).u,  R+- = |V+- - P|,  R0^2 = t0^2 + h^2,
//     f    = ln (R+ + s+)/(R- + s-)                     (written below without cancellation),
//     beta = atan(t0 s+ / (R0^2 + |h| R+)) - atan(t0 s- / (R0^2 + |h| R-)),
//     I_phi = sum_edges (t0 f - |h| beta),   I_E = sgn(h) n sum beta + sum u f.
// Degenerate positions (reading 14): h = 0 drops the beta terms; an edge whose line
// passes through P (R0 = 0) adds nothing to I_phi; P on an edge segment gives an infinite in-plane
// field, as it must.
#pragma once
#include "device_utils.cuh"

namespace bemcub {

struct Vec3 {
  double x, y, z;
};
__device__ __forceinline__ Vec3 vsub(const Vec3& a, const Vec3& b) { return {a.x - b.x, a.y - b.y, a.z - b.z}; }
__device__ __forceinline__ double vdot(const Vec3& a, const Vec3& b) { return a.x * b.x + a.y * b.y + a.z * b.z; }
__device__ __forceinline__ Vec3 vcross(const Vec3& a, const Vec3& b) {
  return {a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x};
}
__device__ __forceinline__ Vec3 vscale(const Vec3& a, double s) { return {a.x * s, a.y * s, a.z * s}; }

// Polygon corners of element `e` in order (3 for a triangle, 4 for a rectangle).
__device__ __forceinline__ int load_polygon(const uint8_t* __restrict__ type, const double* __restrict__ verts, int64_t e,
                                            Vec3 (&V)[4]) {
  const double* v = verts + 9 * e;
  V[0] = {__ldg(v + 0), __ldg(v + 1), __ldg(v + 2)};
  V[1] = {__ldg(v + 3), __ldg(v + 4), __ldg(v + 5)};
  const Vec3 third = {__ldg(v + 6), __ldg(v + 7), __ldg(v + 8)};
  if (__ldg(type + e) == 0) {
    V[2] = third;
    V[3] = third;
    return 3;
  }
  // rectangle P0, P1, P1 + (P3 - P0), P3
  V[2] = {V[1].x + (third.x - V[0].x), V[1].y + (third.y - V[0].y), V[1].z + (third.z - V[0].z)};
  V[3] = third;
  return 4;
}

template <bool WANT_FIELD>
__device__ __noinline__ void analytic_integrals(const Vec3 (&V)[4], int nv, const Vec3& P, double& Iphi, Vec3& IE) {
  Vec3 n = vcross(vsub(V[1], V[0]), vsub(V[nv - 1], V[0]));
  n = vscale(n, 1.0 / sqrt(vdot(n, n)));
  const double h = vdot(n, vsub(P, V[0]));
  const double ah = fabs(h);
  double sphi = 0.0, sbeta = 0.0;
  Vec3 sE = {0.0, 0.0, 0.0};
  Vec3 dm = vsub(V[0], P);
  double Rm = sqrt(vdot(dm, dm));
  for (int i = 0; i < nv; ++i) {
    const int ip = (i + 1 == nv) ? 0 : i + 1;
    const Vec3 dp = vsub(V[ip], P);
    const double Rp = sqrt(vdot(dp, dp));
    Vec3 l = vsub(V[ip], V[i]);
    l = vscale(l, 1.0 / sqrt(vdot(l, l)));
    const Vec3 u = vcross(l, n);
    const double sp = vdot(dp, l), sm = vdot(dm, l), t0 = vdot(dm, u);
    const double R02 = t0 * t0 + h * h;
    // f = ln[(R+ + s+)/(R- + s-)]; (R + s)(R - s) = R0^2 gives the forms free of cancellation
    double f;
    if (sp < 0.0 && sm < 0.0) f = log((Rm - sm) / (Rp - sp));
    else if (sm < 0.0) f = (R02 > 0.0) ? log((Rp + sp) * (Rm - sm) / R02) : CUDART_INF;
    else f = log((Rp + sp) / (Rm + sm));
    if (R02 > 0.0) {
      const double beta = atan(t0 * sp / (R02 + ah * Rp)) - atan(t0 * sm / (R02 + ah * Rm));
      sphi += t0 * f - ah * beta;
      sbeta += beta;
    }
    if (WANT_FIELD) {
      sE.x += u.x * f;
      sE.y += u.y * f;
      sE.z += u.z * f;
    }
    dm = dp;
    Rm = Rp;
  }
  Iphi = sphi;
  if (WANT_FIELD) {
    const double sg = (h > 0.0) ? sbeta : ((h < 0.0) ? -sbeta : 0.0);
    IE = {sE.x + sg * n.x, sE.y + sg * n.y, sE.z + sg * n.z};
  }
}

}  // namespace bemcub
