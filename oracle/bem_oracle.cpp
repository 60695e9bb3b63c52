// ORACLE — TEST INFRASTRUCTURE ONLY.
//
// Plain, slow, obviously-correct CPU implementation of the hot path of arXiv 1606.03743
// (Glueck & Hilk): potential and field of constant-sigma BEM triangles / rectangles by
// Gaussian cubature (Eq. 4.1), the distance-ratio rule choice of Sec. 4 (L159), an analytic
// near-field formula, and the collocation-matrix entries that follow from them.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
// may build, load or call this file.  It shares NO code with the CUDA library
// (paper_1606_03743_b200/csrc): no headers, no tables, no helpers.  The product path never
// routes through it.
//
// Every function cites the passage of /root/reference/PAPER.md it follows.  Arithmetic is
// long double (x87 80-bit) in the parity instantiation; a double instantiation of the very
// same template is what bench.py times as the CPU baseline.  No blocking, fusion or
// reordering beyond the paper's statement: geometry (centroid, area, L) once per element, then
// one field point after the other, elements in index order, the rule's points in table order,
// mapped onto the element for every (element, field point) pair anew (L218).
//
// Parity pins (tests/test_oracle_*.py, all `-m "not gpu"`):
//   tables      : sum w = 1, exact monomial integrals up to the stated degree, failure at d+1
//   mapping     : sum q_i = sigma*A, first moment about the centroid vanishes
//   Eq. 4.1 sum : far-field point-charge limit; closed-form on-axis rectangle potential/field
//                 (also for two triangles tiling the rectangle); uniformly charged sphere;
//                 E = -grad Phi by central differences
//   analytic    : closed forms (square centre, equilateral centroid, on-axis rectangle),
//                 GL2 16 vs 32, long-double adaptive quadrature on tiny inputs
//   pairs       : the single-element integrator (element k seen from point k) against the summed
//                 path on one-element meshes; Duffy-mapped rectangle rules: sum w' = 1, exact
//                 triangle monomials up to (D-1)/2 and not beyond, the printed ~1e-8 at DR = 100 (L169)
//   policy      : the shipped Phi+E distance-ratio limits by the paper's random-element protocol
//   KATRIN Table 1 numbers: parity unpinned (meshes not available).
//
// Build: g++ -O2 -std=c++17 -ffp-contract=off -fopenmp -shared -fPIC bem_oracle.cpp -o liboracle.so
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>
#include <algorithm>
#ifdef _OPENMP
#include <omp.h>
#endif
#include "rule_tables.hpp"

namespace orc {

// CODATA-2018 vacuum permittivity (paper gives no value; DESIGN.md §3 reading 10).
static const long double EPS0 = 8.8541878128e-12L;
static const long double PI_L = 3.14159265358979323846264338327950288L;
inline long double coulomb_k() { return 1.0L / (4.0L * PI_L * EPS0); }

enum { TRI = 0, RECT = 1 };
enum { ERR_OK = 0, ERR_INVALID = -1, ERR_DEGENERATE = -2, ERR_NOT_RECT = -3, ERR_BAD_RULE = -4 };

template <class T> inline T tsqrt(T x);
template <> inline long double tsqrt(long double x) { return sqrtl(x); }
template <> inline double tsqrt(double x) { return sqrt(x); }
template <class T> inline T tlog(T x);
template <> inline long double tlog(long double x) { return logl(x); }
template <> inline double tlog(double x) { return log(x); }
template <class T> inline T tatan(T x);
template <> inline long double tatan(long double x) { return atanl(x); }
template <> inline double tatan(double x) { return atan(x); }
template <class T> inline T tabs(T x) { return x < 0 ? -x : x; }

inline int threads_for(int nthreads) {
#ifdef _OPENMP
    return nthreads > 0 ? nthreads : omp_get_max_threads();
#else
    (void)nthreads;
    return 1;
#endif
}

template <class T> struct V3 { T x, y, z; };
template <class T> inline V3<T> sub(const V3<T>& a, const V3<T>& b) { return {a.x - b.x, a.y - b.y, a.z - b.z}; }
template <class T> inline T dot(const V3<T>& a, const V3<T>& b) { return a.x * b.x + a.y * b.y + a.z * b.z; }
template <class T> inline V3<T> cross(const V3<T>& a, const V3<T>& b) {
    return {a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x};
}
template <class T> inline T norm(const V3<T>& a) { return tsqrt<T>(dot(a, a)); }

// ---------------------------------------------------------------------------------------
// Geometry of one element.  Triangle: vertices A,B,C (Eq. 3.3).  Rectangle: corner
// P0, P1 = P0 + a u_x, P3 = P0 + b u_y; centre, side lengths and side unit vectors as in
// Eq. 3.2 (L101-105).  L = average side length (L66): (a+b+c)/3 for the triangle, (a+b)/2
// for the rectangle (DESIGN.md §3 reading 6).
template <class T> struct Geom {
    int type;
    V3<T> v[4];     // polygon vertices in order (3 or 4)
    int nv;
    V3<T> cen;      // Q_cen
    T area;         // script-A
    T L;            // average side length
    V3<T> hx, hy;   // rectangle: (a/2) u_x, (b/2) u_y
};

template <class T>
int make_geom(int type, const double* vv, Geom<T>& g) {
    V3<T> p0{(T)vv[0], (T)vv[1], (T)vv[2]}, p1{(T)vv[3], (T)vv[4], (T)vv[5]}, p2{(T)vv[6], (T)vv[7], (T)vv[8]};
    g.type = type;
    if (type == TRI) {
        g.nv = 3;
        g.v[0] = p0; g.v[1] = p1; g.v[2] = p2;
        V3<T> e1 = sub(p1, p0), e2 = sub(p2, p0);
        g.area = (T)0.5 * norm(cross(e1, e2));
        g.cen = {(p0.x + p1.x + p2.x) / (T)3, (p0.y + p1.y + p2.y) / (T)3, (p0.z + p1.z + p2.z) / (T)3};
        g.L = (norm(sub(p1, p0)) + norm(sub(p2, p1)) + norm(sub(p0, p2))) / (T)3;
        g.hx = g.hy = {0, 0, 0};
        if (!(g.area > 0)) return ERR_DEGENERATE;
    } else if (type == RECT) {
        g.nv = 4;
        V3<T> e1 = sub(p1, p0), e2 = sub(p2, p0);
        T a = norm(e1), b = norm(e2);
        if (!(a > 0) || !(b > 0)) return ERR_DEGENERATE;
        if (tabs(dot(e1, e2)) > (T)1e-12 * a * b) return ERR_NOT_RECT;
        g.v[0] = p0; g.v[1] = p1;
        g.v[2] = {p1.x + e2.x, p1.y + e2.y, p1.z + e2.z};
        g.v[3] = p2;
        g.area = a * b;
        g.cen = {p0.x + (T)0.5 * e1.x + (T)0.5 * e2.x, p0.y + (T)0.5 * e1.y + (T)0.5 * e2.y,
                 p0.z + (T)0.5 * e1.z + (T)0.5 * e2.z};
        g.L = (a + b) / (T)2;
        // (a/2) u_x = e1/2, (b/2) u_y = e2/2
        g.hx = {(T)0.5 * e1.x, (T)0.5 * e1.y, (T)0.5 * e1.z};
        g.hy = {(T)0.5 * e2.x, (T)0.5 * e2.y, (T)0.5 * e2.z};
    } else {
        return ERR_INVALID;
    }
    return ERR_OK;
}

// ---------------------------------------------------------------------------------------
// Gaussian points Q_i and relative weights w_i of one element for one rule level.
// Triangle: Q = lA*A + lB*B + lC*C (Eq. 3.3).  Rectangle: Q = Q_cen + (a/2) x u_x +
// (b/2) y u_y (Eq. 3.2).
template <class T> struct Pt { T x, y, z, w; };

template <class T>
void element_points(const Geom<T>& g, int level, std::vector<Pt<T>>& out) {
    out.clear();
    if (g.type == TRI) {
        for (const TriNode& nd : tri_rule(level)) {
            T la = (T)nd.la, lb = (T)nd.lb, lc = (T)nd.lc;
            out.push_back({la * g.v[0].x + lb * g.v[1].x + lc * g.v[2].x,
                           la * g.v[0].y + lb * g.v[1].y + lc * g.v[2].y,
                           la * g.v[0].z + lb * g.v[1].z + lc * g.v[2].z, (T)nd.w});
        }
    } else {
        for (const RectNode& nd : rect_rule(level)) {
            T x = (T)nd.x, y = (T)nd.y;
            out.push_back({g.cen.x + x * g.hx.x + y * g.hy.x, g.cen.y + x * g.hx.y + y * g.hy.y,
                           g.cen.z + x * g.hx.z + y * g.hy.z, (T)nd.w});
        }
    }
}

// ---------------------------------------------------------------------------------------
// Duffy variant (Sec. 4): "a triangle can be mapped into a rectangle by the Duffy
// transformation, therefore the numerical integration over a triangle by Gaussian cubature can also
// be done by using the Duffy transformation in conjunction with the Gaussian cubature formulas for
// rectangles of App. B".  The paper prints no formula (Refs. [64,69]); reading 20 takes
// the classical map that collapses one edge of the square onto vertex A:
//     Q(u,v) = A + u [ (B - A) + v (C - B) ],  (u,v) in [0,1]^2,   dS = 2 area u du dv,
// with the collapsing coordinate along the rule's y axis: u = (1+y)/2, v = (1+x)/2 for a node
// (x,y) of the rectangle rule.  (Tables B2, B4, B5 are not symmetric under x <-> y; of the two
// assignments this one reproduces the error the paper prints for the 7-point rule at DR = 100,
// "about 1e-8" (L169): 6e-9 against 7e-11 for the other.)  Relative to the triangle area the
// node weight becomes w' = 2 u w = (1 + y) w  (sum w' = 1 because the rule integrates y exactly).
// A triangle polynomial of degree d becomes a polynomial of degree up to 2d in (u,v), times the
// Jacobian u: exactness is guaranteed for d <= (D - 1)/2 only, D the degree of the rectangle rule.
template <class T>
void element_points_duffy(const Geom<T>& g, int level, std::vector<Pt<T>>& out) {
    out.clear();
    const V3<T> AB = sub(g.v[1], g.v[0]), BC = sub(g.v[2], g.v[1]);
    for (const RectNode& nd : rect_rule(level)) {
        const T u = ((T)1 + (T)nd.y) / (T)2, v = ((T)1 + (T)nd.x) / (T)2;
        out.push_back({g.v[0].x + u * (AB.x + v * BC.x), g.v[0].y + u * (AB.y + v * BC.y),
                       g.v[0].z + u * (AB.z + v * BC.z), ((T)1 + (T)nd.y) * (T)nd.w});
    }
}

// ---------------------------------------------------------------------------------------
// Analytic near-field integrals of a flat polygon (the paper cites but does not print its
// analytic formulas, L68/L78; DESIGN.md §3 reading 9 takes this exact closed form of
// Eq. 2.1, a line-integral form of the same family as Ref. [27]):
//   I_phi = Int dS / R,  I_E = Int dS (P-Q)/R^3     (unit sigma, no 1/(4 pi eps0))
// With n the unit normal, h = n.(P - V0), and per edge V- -> V+:
//   l = unit edge vector, u = l x n (outward in-plane normal), s+- = (V+- - P).l,
//   t0 = (V- - P).u, R+- = |P - V+-|, R0^2 = t0^2 + h^2,
//   f  = ln[(R+ + s+)/(R- + s-)] written in the cancellation-free equivalent form for the
//        sign pattern of s+-,
//   beta = atan(t0 s+ /(R0^2 + |h| R+)) - atan(t0 s- /(R0^2 + |h| R-)),
//   I_phi = sum_i (t0 f - |h| beta),  I_E = sgn(h) n sum_i beta + sum_i u f.
// An edge whose line contains P (R0 = 0) contributes 0 to I_phi; its f is finite unless P
// lies on the edge segment itself (then the in-plane field is log-singular: inf).
template <class T>
void analytic_integrals(const Geom<T>& g, const V3<T>& P, T& Iphi, V3<T>& IE) {
    V3<T> nrm = cross(sub(g.v[1], g.v[0]), sub(g.v[g.nv - 1], g.v[0]));
    T nn = norm(nrm);
    nrm = {nrm.x / nn, nrm.y / nn, nrm.z / nn};
    T h = dot(nrm, sub(P, g.v[0]));
    T ah = tabs(h);
    T sg = (h > 0) ? (T)1 : ((h < 0) ? (T)-1 : (T)0);
    Iphi = 0;
    T sumbeta = 0;
    IE = {0, 0, 0};
    for (int i = 0; i < g.nv; ++i) {
        const V3<T>& Vm = g.v[i];
        const V3<T>& Vp = g.v[(i + 1) % g.nv];
        V3<T> l = sub(Vp, Vm);
        T len = norm(l);
        l = {l.x / len, l.y / len, l.z / len};
        V3<T> u = cross(l, nrm);
        V3<T> dm = sub(Vm, P), dp = sub(Vp, P);
        T sp = dot(dp, l), sm = dot(dm, l), t0 = dot(dm, u);
        T Rp = norm(dp), Rm = norm(dm);
        T R02 = t0 * t0 + h * h;
        T f, beta = 0;
        if (sp < 0 && sm < 0)        f = tlog<T>((Rm - sm) / (Rp - sp));
        else if (sm < 0) {           // s- < 0 <= s+ : R- + s- = R0^2 / (R- - s-)
            if (R02 > 0) f = tlog<T>((Rp + sp) * (Rm - sm) / R02);
            else         f = (T)INFINITY;                 // P on the edge segment
        } else                       f = tlog<T>((Rp + sp) / (Rm + sm));
        if (R02 > 0) {
            beta = tatan<T>(t0 * sp / (R02 + ah * Rp)) - tatan<T>(t0 * sm / (R02 + ah * Rm));
            Iphi += t0 * f - ah * beta;
        }
        sumbeta += beta;
        IE.x += u.x * f; IE.y += u.y * f; IE.z += u.z * f;
    }
    IE.x += sg * nrm.x * sumbeta; IE.y += sg * nrm.y * sumbeta; IE.z += sg * nrm.z * sumbeta;
}

// ---------------------------------------------------------------------------------------
// Gauss-Legendre nodes on [-1,1] by Newton iteration on P_n (used by GL2 and by the adaptive
// reference).  Textbook; pinned in the tests by exact polynomial integration.
static void gauss_legendre(int n, std::vector<long double>& x, std::vector<long double>& w) {
    x.resize(n); w.resize(n);
    for (int i = 0; i < n; ++i) {
        long double z = cosl(PI_L * (i + 0.75L) / (n + 0.5L));
        long double pp = 1;
        for (int it = 0; it < 100; ++it) {
            long double p1 = 1, p2 = 0;
            for (int j = 1; j <= n; ++j) {
                long double p3 = p2; p2 = p1;
                p1 = ((2 * j - 1) * z * p2 - (j - 1) * p3) / j;
            }
            pp = n * (z * p1 - p2) / (z * z - 1);
            long double dz = p1 / pp;
            z -= dz;
            if (fabsl(dz) < 1e-21L) break;
        }
        // recompute derivative at converged z
        long double p1 = 1, p2 = 0;
        for (int j = 1; j <= n; ++j) { long double p3 = p2; p2 = p1; p1 = ((2 * j - 1) * z * p2 - (j - 1) * p3) / j; }
        pp = n * (z * p1 - p2) / (z * z - 1);
        x[i] = z;
        w[i] = 2 / ((1 - z * z) * pp * pp);
    }
}

struct F4 { long double v[4]; };

// integrand of Eq. 2.1 (L64) at surface point Q, times the area Jacobian jac
static inline void coulomb_integrand(const V3<long double>& P, const V3<long double>& Q, long double jac, F4& acc) {
    V3<long double> d = sub(P, Q);
    long double r2 = dot(d, d), r = sqrtl(r2), i3 = jac / (r2 * r);
    acc.v[0] += jac / r; acc.v[1] += d.x * i3; acc.v[2] += d.y * i3; acc.v[3] += d.z * i3;
}

// surface point and Jacobian for parameters (s,t) in [0,1]^2.
// Rectangle: x = 2s-1, y = 2t-1 in Eq. 3.2, dS = area ds dt.
// Triangle: collapsed map Q = A + s(B-A) + t(1-s)(C-A), dS = 2*area*(1-s) ds dt.
static inline void surface_point(const Geom<long double>& g, long double s, long double t,
                                 V3<long double>& Q, long double& jac) {
    if (g.type == RECT) {
        long double x = 2 * s - 1, y = 2 * t - 1;
        Q = {g.cen.x + x * g.hx.x + y * g.hy.x, g.cen.y + x * g.hx.y + y * g.hy.y, g.cen.z + x * g.hx.z + y * g.hy.z};
        jac = g.area;
    } else {
        V3<long double> e1 = sub(g.v[1], g.v[0]), e2 = sub(g.v[2], g.v[0]);
        long double c = t * (1 - s);
        Q = {g.v[0].x + s * e1.x + c * e2.x, g.v[0].y + s * e1.y + c * e2.y, g.v[0].z + s * e1.z + c * e2.z};
        jac = 2 * g.area * (1 - s);
    }
}

// GL2: two successive one-dimensional Gauss-Legendre quadratures with n nodes each (L40, L78).
static void gl2_integrals(const Geom<long double>& g, const V3<long double>& P, int n, F4& out) {
    std::vector<long double> x, w;
    gauss_legendre(n, x, w);
    out = F4{{0, 0, 0, 0}};
    for (int i = 0; i < n; ++i) {
        F4 inner{{0, 0, 0, 0}};
        long double s = 0.5L * (x[i] + 1);
        for (int j = 0; j < n; ++j) {
            long double t = 0.5L * (x[j] + 1), jac;
            V3<long double> Q;
            surface_point(g, s, t, Q, jac);
            coulomb_integrand(P, Q, jac * 0.25L * w[j], inner);
        }
        for (int k = 0; k < 4; ++k) out.v[k] += w[i] * inner.v[k];
    }
}

// Adaptive reference: nested 1-D adaptive bisection, each panel integrated with GL-12 and
// accepted when it agrees with the sum of its two half panels (brute force for tiny inputs).
struct Adaptive {
    const Geom<long double>& g;
    V3<long double> P;
    std::vector<long double> x, w;
    long double scale[4];
    long double tol;
    long double err;
    Adaptive(const Geom<long double>& g_, const V3<long double>& P_, long double tol_) : g(g_), P(P_), tol(tol_), err(0) {
        gauss_legendre(12, x, w);
    }
    F4 inner_panel(long double s, long double a, long double b) const {
        F4 r{{0, 0, 0, 0}};
        for (size_t j = 0; j < x.size(); ++j) {
            long double t = 0.5L * ((b - a) * x[j] + (a + b)), jac;
            V3<long double> Q;
            surface_point(g, s, t, Q, jac);
            coulomb_integrand(P, Q, jac * 0.5L * (b - a) * w[j], r);
        }
        return r;
    }
    bool close(const F4& a, const F4& b, long double frac, long double t) const {
        for (int k = 0; k < 4; ++k)
            if (fabsl(a.v[k] - b.v[k]) > t * frac * scale[k]) return false;
        return true;
    }
    F4 inner_rec(long double s, long double a, long double b, const F4& whole, int depth) const {
        long double m = 0.5L * (a + b);
        F4 l = inner_panel(s, a, m), r = inner_panel(s, m, b), sum;
        for (int k = 0; k < 4; ++k) sum.v[k] = l.v[k] + r.v[k];
        if (depth > 48 || close(whole, sum, b - a, tol * 0.1L)) return sum;
        F4 L2 = inner_rec(s, a, m, l, depth + 1), R2 = inner_rec(s, m, b, r, depth + 1);
        for (int k = 0; k < 4; ++k) sum.v[k] = L2.v[k] + R2.v[k];
        return sum;
    }
    F4 inner(long double s) const { return inner_rec(s, 0, 1, inner_panel(s, 0, 1), 0); }
    F4 outer_panel(long double a, long double b) const {
        F4 r{{0, 0, 0, 0}};
        for (size_t i = 0; i < x.size(); ++i) {
            long double s = 0.5L * ((b - a) * x[i] + (a + b));
            F4 in = inner(s);
            for (int k = 0; k < 4; ++k) r.v[k] += 0.5L * (b - a) * w[i] * in.v[k];
        }
        return r;
    }
    F4 outer_rec(long double a, long double b, const F4& whole, int depth) {
        long double m = 0.5L * (a + b);
        F4 l = outer_panel(a, m), r = outer_panel(m, b), sum;
        for (int k = 0; k < 4; ++k) sum.v[k] = l.v[k] + r.v[k];
        if (depth > 48 || close(whole, sum, b - a, tol)) {
            for (int k = 0; k < 4; ++k) err = std::max(err, fabsl(whole.v[k] - sum.v[k]) / scale[k]);
            return sum;
        }
        F4 L2 = outer_rec(a, m, l, depth + 1), R2 = outer_rec(m, b, r, depth + 1);
        for (int k = 0; k < 4; ++k) sum.v[k] = L2.v[k] + R2.v[k];
        return sum;
    }
    F4 run() {
        F4 est;
        gl2_integrals(g, P, 16, est);
        scale[0] = fabsl(est.v[0]);
        long double e = sqrtl(est.v[1] * est.v[1] + est.v[2] * est.v[2] + est.v[3] * est.v[3]);
        // field scale: never smaller than potential/distance so that symmetric zeros do not stall
        long double D = norm(sub(P, g.cen));
        scale[1] = scale[2] = scale[3] = std::max(e, scale[0] / std::max(D, g.L));
        return outer_rec(0, 1, outer_panel(0, 1), 0);
    }
};

// ---------------------------------------------------------------------------------------
// Distance-ratio rule choice (L66, L159).  dr[type][0..4] = upper DR limits of
// {analytic, N=33, N=19|17, N=12, N=7}; N=4 above dr[type][4].  Bands are lower-inclusive
// (DESIGN.md §3 reading 8).  The decision is taken in double precision by comparing D^2 with
// (limit*L)^2.  Returns 0..4 = rule level (N = 4,7,12,19|17,33), 5 = analytic.
// levels_mask: bit k enables level k, bit 5 enables the analytic branch; a disabled choice
// moves to the next more accurate enabled one (and, if none, to the most accurate enabled).
static int choose_level(double D2, double L, const double* dr5, int levels_mask) {
    int want = 0;                                 // band -> level: band 0 = analytic (5), 1 -> 4, 2 -> 3, 3 -> 2, 4 -> 1
    for (int b = 0; b < 5; ++b) {
        double thr = dr5[b] * L;
        if (D2 < thr * thr) { want = (b == 0) ? 5 : 5 - b; break; }
    }
    for (int lv = want; lv <= 5; ++lv)
        if (levels_mask & (1 << lv)) return lv;
    for (int lv = want - 1; lv >= 0; --lv)
        if (levels_mask & (1 << lv)) return lv;
    return -1;
}

// ---------------------------------------------------------------------------------------
// Eq. 4.1 (L139-143): Phi(P) = k sum q_i / |P-Q_i|,  E(P) = k sum q_i (P-Q_i)/|P-Q_i|^3,
// q_i = w_i sigma A; summed over all elements for each field point (L34, L202).
template <class T>
int eval_impl(int64_t n, const uint8_t* etype, const double* verts, const double* sigma, int level,
              const double* dr, int levels_mask, int64_t m, const double* pts, double* phi, double* E,
              double* Sphi, double* SE, int64_t* npi, int64_t* nana, int nthreads) {
    if (n < 0 || m < 0) return ERR_INVALID;
    if (level < -1 || level > 4) return ERR_BAD_RULE;
    if (level == -1 && (!dr || (levels_mask & 63) == 0)) return ERR_INVALID;
    // step 2 (geometry) once per element
    std::vector<Geom<T>> G((size_t)n);
    for (int64_t e = 0; e < n; ++e) {
        int rc = make_geom<T>(etype[e], verts + 9 * e, G[e]);
        if (rc) return rc;
    }
    const T k = (T)coulomb_k();
    // steps 3-5, one field point after the other: elements in index order, the rule's points in table order
    // (nthreads > 0 limits this call only; it does not change the process-wide OpenMP setting)
    const int nt = threads_for(nthreads);
#pragma omp parallel for schedule(dynamic, 1) num_threads(nt)
    for (int64_t j = 0; j < m; ++j) {
        const V3<T> P{(T)pts[3 * j], (T)pts[3 * j + 1], (T)pts[3 * j + 2]};
        T aphi = 0, aex = 0, aey = 0, aez = 0, asphi = 0, ase = 0;
        int64_t cnt = 0, cana = 0;
        std::vector<Pt<T>> pv;
        for (int64_t e = 0; e < n; ++e) {
            const Geom<T>& g = G[e];
            int lv = level;
            if (level == -1) {
                const double dx = pts[3 * j] - (double)g.cen.x, dy = pts[3 * j + 1] - (double)g.cen.y, dz = pts[3 * j + 2] - (double)g.cen.z;
                lv = choose_level(dx * dx + dy * dy + dz * dz, (double)g.L, dr + 5 * g.type, levels_mask);
            }
            if (lv == 5) {
                T Ip; V3<T> Ie;
                analytic_integrals<T>(g, P, Ip, Ie);
                const T s = (T)sigma[e];
                aphi += s * Ip; aex += s * Ie.x; aey += s * Ie.y; aez += s * Ie.z;
                asphi += tabs(s * Ip);
                ase += tabs(s) * norm(Ie);
                ++cana;
                continue;
            }
            element_points<T>(g, lv, pv);
            const T q = (T)sigma[e] * g.area;               // q = sigma * A (L143)
            for (const Pt<T>& p : pv) {
                const T qi = p.w * q;                        // q_i = w_i q (L143)
                const T dx = P.x - p.x, dy = P.y - p.y, dz = P.z - p.z;
                const T r2 = dx * dx + dy * dy + dz * dz;
                const T inv = (T)1 / tsqrt<T>(r2);           // one square root, one division (L46)
                const T inv3 = inv * inv * inv;
                aphi += qi * inv;
                aex += qi * dx * inv3; aey += qi * dy * inv3; aez += qi * dz * inv3;
                asphi += tabs(qi) * inv;
                ase += tabs(qi) * inv * inv;
            }
            cnt += (int64_t)pv.size();
        }
        if (phi) phi[j] = (double)(k * aphi);
        if (E) { E[3 * j] = (double)(k * aex); E[3 * j + 1] = (double)(k * aey); E[3 * j + 2] = (double)(k * aez); }
        if (Sphi) Sphi[j] = (double)(k * asphi);
        if (SE) SE[j] = (double)(k * ase);
        if (npi) npi[j] = cnt;
        if (nana) nana[j] = cana;
    }
    return ERR_OK;
}

// ---------------------------------------------------------------------------------------
// Field gradient from the same point charges (L273: "higher derivatives of the field ... can be
// easily computed from the point charges"): differentiating the E-term of Eq. 4.1 (L141),
//     G_ij(P) = dE_i/dx_j = k sum q_i [ delta_ij / r^3 - 3 d_i d_j / r^5 ],   d = P - Q_i, r = |d|.
// Output order per field point: xx, yy, zz, xy, xz, yz (G is symmetric, and traceless away from
// the charges).  SG = k sum |q_i| / r^3 is the parity denominator.  Cubature levels only: the
// paper gives no analytic expression for derivatives, so levels_mask must not contain bit 5.
template <class T>
int grad_impl(int64_t n, const uint8_t* etype, const double* verts, const double* sigma, int level,
              const double* dr, int levels_mask, int64_t m, const double* pts, double* G, double* SG) {
    if (n < 0 || m < 0 || !G) return ERR_INVALID;
    if (level < -1 || level > 4) return ERR_BAD_RULE;
    if (level == -1 && (!dr || (levels_mask & 31) == 0 || (levels_mask & 32))) return ERR_INVALID;
    for (int64_t e = 0; e < n; ++e) {
        Geom<T> g;
        int rc = make_geom<T>(etype[e], verts + 9 * e, g);
        if (rc) return rc;
    }
    const T k = (T)coulomb_k();
#pragma omp parallel for schedule(dynamic, 4)
    for (int64_t j = 0; j < m; ++j) {
        const V3<T> P{(T)pts[3 * j], (T)pts[3 * j + 1], (T)pts[3 * j + 2]};
        T a[6] = {0, 0, 0, 0, 0, 0}, sg = 0;
        std::vector<Pt<T>> pv;
        for (int64_t e = 0; e < n; ++e) {
            Geom<T> g;
            make_geom<T>(etype[e], verts + 9 * e, g);
            int lv = level;
            if (level == -1) {
                double dx = pts[3 * j] - (double)g.cen.x, dy = pts[3 * j + 1] - (double)g.cen.y, dz = pts[3 * j + 2] - (double)g.cen.z;
                lv = choose_level(dx * dx + dy * dy + dz * dz, (double)g.L, dr + 5 * g.type, levels_mask);
            }
            element_points<T>(g, lv, pv);
            const T q = (T)sigma[e] * g.area;
            for (const Pt<T>& p : pv) {
                const T qi = p.w * q;
                const T dx = P.x - p.x, dy = P.y - p.y, dz = P.z - p.z;
                const T r2 = dx * dx + dy * dy + dz * dz;
                const T inv = (T)1 / tsqrt<T>(r2);
                const T inv3 = inv * inv * inv, inv5 = inv3 * inv * inv;
                a[0] += qi * (inv3 - 3 * dx * dx * inv5);
                a[1] += qi * (inv3 - 3 * dy * dy * inv5);
                a[2] += qi * (inv3 - 3 * dz * dz * inv5);
                a[3] += qi * (-3 * dx * dy * inv5);
                a[4] += qi * (-3 * dx * dz * inv5);
                a[5] += qi * (-3 * dy * dz * inv5);
                sg += tabs(qi) * inv3;
            }
        }
        for (int c = 0; c < 6; ++c) G[6 * j + c] = (double)(k * a[c]);
        if (SG) SG[j] = (double)(k * sg);
    }
    return ERR_OK;
}

// ---------------------------------------------------------------------------------------
// Non-constant charge density (L275: "linear, quadratic etc. ... q_i = w_i A sigma(Q_i)"): sigma
// varies linearly over the element, given by its values sv[3] at the three stored vertices
// (triangle A,B,C; rectangle P0,P1,P3 - the fourth corner then carries sv[1]+sv[2]-sv[0]).
// sigma(Q) is evaluated from the POSITION of the Gaussian point (in-plane coordinates by a 2x2
// least-squares solve), not from the rule's reference coordinates.  Cubature levels only.
template <class T>
inline T sigma_at(const double* v9, const double* sv, const Pt<T>& Q) {
    const V3<T> A{(T)v9[0], (T)v9[1], (T)v9[2]}, B{(T)v9[3], (T)v9[4], (T)v9[5]}, Cc{(T)v9[6], (T)v9[7], (T)v9[8]};
    const V3<T> e1 = sub(B, A), e2 = sub(Cc, A), d = sub(V3<T>{Q.x, Q.y, Q.z}, A);
    const T a11 = dot(e1, e1), a12 = dot(e1, e2), a22 = dot(e2, e2), b1 = dot(d, e1), b2 = dot(d, e2);
    const T det = a11 * a22 - a12 * a12;
    const T s = (b1 * a22 - b2 * a12) / det, t = (a11 * b2 - a12 * b1) / det;
    return (T)sv[0] + s * ((T)sv[1] - (T)sv[0]) + t * ((T)sv[2] - (T)sv[0]);
}

template <class T>
int linear_impl(int64_t n, const uint8_t* etype, const double* verts, const double* sigma_v, int level,
                const double* dr, int levels_mask, int64_t m, const double* pts, double* phi, double* E,
                double* Sphi, double* SE) {
    if (n < 0 || m < 0) return ERR_INVALID;
    if (level < -1 || level > 4) return ERR_BAD_RULE;
    if (level == -1 && (!dr || (levels_mask & 31) == 0 || (levels_mask & 32))) return ERR_INVALID;
    for (int64_t e = 0; e < n; ++e) {
        Geom<T> g;
        int rc = make_geom<T>(etype[e], verts + 9 * e, g);
        if (rc) return rc;
    }
    const T k = (T)coulomb_k();
#pragma omp parallel for schedule(dynamic, 4)
    for (int64_t j = 0; j < m; ++j) {
        const V3<T> P{(T)pts[3 * j], (T)pts[3 * j + 1], (T)pts[3 * j + 2]};
        T aphi = 0, ax = 0, ay = 0, az = 0, sphi = 0, se = 0;
        std::vector<Pt<T>> pv;
        for (int64_t e = 0; e < n; ++e) {
            Geom<T> g;
            make_geom<T>(etype[e], verts + 9 * e, g);
            int lv = level;
            if (level == -1) {
                double dx = pts[3 * j] - (double)g.cen.x, dy = pts[3 * j + 1] - (double)g.cen.y, dz = pts[3 * j + 2] - (double)g.cen.z;
                lv = choose_level(dx * dx + dy * dy + dz * dz, (double)g.L, dr + 5 * g.type, levels_mask);
            }
            element_points<T>(g, lv, pv);
            for (const Pt<T>& p : pv) {
                const T qi = p.w * g.area * sigma_at<T>(verts + 9 * e, sigma_v + 3 * e, p);   // q_i = w_i A sigma(Q_i)
                const T dx = P.x - p.x, dy = P.y - p.y, dz = P.z - p.z;
                const T inv = (T)1 / tsqrt<T>(dx * dx + dy * dy + dz * dz);
                const T inv3 = inv * inv * inv;
                aphi += qi * inv;
                ax += qi * dx * inv3; ay += qi * dy * inv3; az += qi * dz * inv3;
                sphi += tabs(qi) * inv;
                se += tabs(qi) * inv * inv;
            }
        }
        if (phi) phi[j] = (double)(k * aphi);
        if (E) { E[3 * j] = (double)(k * ax); E[3 * j + 1] = (double)(k * ay); E[3 * j + 2] = (double)(k * az); }
        if (Sphi) Sphi[j] = (double)(k * sphi);
        if (SE) SE[j] = (double)(k * se);
    }
    return ERR_OK;
}

// ---------------------------------------------------------------------------------------
// The single-element boundary integrator (the paper's innermost layer, L193-196 item a): element k
// seen from field point k, k < K, no sum over elements.  This is the unit of the paper's accuracy
// protocol (L68, L149: 1000 random elements and directions per distance ratio).
// method: 0..4 cubature level (Eq. 4.1 with the element's own rule); 5 the analytic closed form;
//         -1 the distance-ratio choice (dr, levels_mask); 8+l (l = 0..4) the rectangle rule of
//         level l - on a triangle through the Duffy map above, on a rectangle as it is.
// used[k] (may be null) = what was evaluated: 0..4, 5 = analytic.
template <class T>
int pairs_impl(int64_t K, const uint8_t* etype, const double* verts, const double* sigma, int method,
               const double* dr, int levels_mask, const double* pts, double* phi, double* E, double* Sphi,
               double* SE, uint8_t* used) {
    if (K < 0) return ERR_INVALID;
    if (!(method >= -1 && method <= 5) && !(method >= 8 && method <= 12)) return ERR_BAD_RULE;
    if (method == -1 && (!dr || (levels_mask & 63) == 0)) return ERR_INVALID;
    for (int64_t e = 0; e < K; ++e) {
        Geom<T> g;
        int rc = make_geom<T>(etype[e], verts + 9 * e, g);
        if (rc) return rc;
    }
    const T k = (T)coulomb_k();
#pragma omp parallel for schedule(static)
    for (int64_t e = 0; e < K; ++e) {
        Geom<T> g;
        make_geom<T>(etype[e], verts + 9 * e, g);
        const V3<T> P{(T)pts[3 * e], (T)pts[3 * e + 1], (T)pts[3 * e + 2]};
        const T sg = sigma ? (T)sigma[e] : (T)1;
        int lv = method;
        if (method == -1) {
            const double dx = pts[3 * e] - (double)g.cen.x, dy = pts[3 * e + 1] - (double)g.cen.y, dz = pts[3 * e + 2] - (double)g.cen.z;
            lv = choose_level(dx * dx + dy * dy + dz * dz, (double)g.L, dr + 5 * g.type, levels_mask);
        }
        T aphi = 0, ax = 0, ay = 0, az = 0, sphi = 0, se = 0;
        if (lv == 5) {
            T Ip; V3<T> Ie;
            analytic_integrals<T>(g, P, Ip, Ie);
            aphi = sg * Ip; ax = sg * Ie.x; ay = sg * Ie.y; az = sg * Ie.z;
            sphi = tabs(sg * Ip); se = tabs(sg) * norm(Ie);
        } else {
            std::vector<Pt<T>> pv;
            if (lv >= 8 && g.type == TRI) element_points_duffy<T>(g, lv - 8, pv);
            else element_points<T>(g, lv >= 8 ? lv - 8 : lv, pv);
            const T q = sg * g.area;
            for (const Pt<T>& p : pv) {
                const T qi = p.w * q;
                const T dx = P.x - p.x, dy = P.y - p.y, dz = P.z - p.z;
                const T inv = (T)1 / tsqrt<T>(dx * dx + dy * dy + dz * dz);
                const T inv3 = inv * inv * inv;
                aphi += qi * inv;
                ax += qi * dx * inv3; ay += qi * dy * inv3; az += qi * dz * inv3;
                sphi += tabs(qi) * inv;
                se += tabs(qi) * inv * inv;
            }
        }
        if (phi) phi[e] = (double)(k * aphi);
        if (E) { E[3 * e] = (double)(k * ax); E[3 * e + 1] = (double)(k * ay); E[3 * e + 2] = (double)(k * az); }
        if (Sphi) Sphi[e] = (double)(k * sphi);
        if (SE) SE[e] = (double)(k * se);
        if (used) used[e] = (uint8_t)(lv >= 8 ? lv - 8 : lv);
    }
    return ERR_OK;
}

}  // namespace orc

using namespace orc;

extern "C" {

double orc_coulomb_k() { return (double)coulomb_k(); }

int orc_rule_info(int etype, int level, int* npts, int* degree) {
    if (level < 0 || level > 4 || (etype != TRI && etype != RECT)) return ERR_BAD_RULE;
    if (etype == TRI) { if (npts) *npts = (int)tri_rule(level).size(); if (degree) *degree = tri_degree(level); }
    else              { if (npts) *npts = (int)rect_rule(level).size(); if (degree) *degree = rect_degree(level); }
    return ERR_OK;
}

// coords: triangle [N][3] barycentric, rectangle [N][2] natural; w: [N]
int orc_rule_nodes(int etype, int level, double* coords, double* w) {
    if (level < 0 || level > 4 || (etype != TRI && etype != RECT)) return ERR_BAD_RULE;
    if (etype == TRI) {
        auto r = tri_rule(level);
        for (size_t i = 0; i < r.size(); ++i) { coords[3 * i] = (double)r[i].la; coords[3 * i + 1] = (double)r[i].lb; coords[3 * i + 2] = (double)r[i].lc; w[i] = (double)r[i].w; }
    } else {
        auto r = rect_rule(level);
        for (size_t i = 0; i < r.size(); ++i) { coords[2 * i] = (double)r[i].x; coords[2 * i + 1] = (double)r[i].y; w[i] = (double)r[i].w; }
    }
    return ERR_OK;
}

// The residual |sum_i w_i m(Q_i) - exact| of monomial integration, evaluated in long double
// (reference triangle (0,0),(1,0),(0,1): x^a y^b, exact a! b! 2/(a+b+2)! ; square [-1,1]^2:
// x^a y^b, exact 1/((a+1)(b+1)) for even a,b else 0 — all relative to the area).  L113.
double orc_rule_monomial_residual(int etype, int level, int a, int b) {
    long double s = 0, exact;
    if (etype == TRI) {
        for (const TriNode& nd : tri_rule(level)) s += nd.w * powl(nd.lb, a) * powl(nd.lc, b);
        long double num = 2;
        for (int i = 2; i <= a; ++i) num *= i;
        for (int i = 2; i <= b; ++i) num *= i;
        long double den = 1;
        for (int i = 2; i <= a + b + 2; ++i) den *= i;
        exact = num / den;
    } else {
        for (const RectNode& nd : rect_rule(level)) s += nd.w * powl(nd.x, a) * powl(nd.y, b);
        exact = (a % 2 == 0 && b % 2 == 0) ? 1.0L / ((a + 1) * (b + 1)) : 0.0L;
    }
    return (double)(s - exact);
}

int orc_geometry(int64_t n, const uint8_t* etype, const double* verts, double* cen, double* area, double* L) {
    for (int64_t e = 0; e < n; ++e) {
        Geom<long double> g;
        int rc = make_geom<long double>(etype[e], verts + 9 * e, g);
        if (rc) return rc;
        if (cen) { cen[3 * e] = (double)g.cen.x; cen[3 * e + 1] = (double)g.cen.y; cen[3 * e + 2] = (double)g.cen.z; }
        if (area) area[e] = (double)g.area;
        if (L) L[e] = (double)g.L;
    }
    return ERR_OK;
}

// Expanded point charges of all elements for one rule level: xyzq[sumN][4] = (Q_i, q_i = w_i sigma A).
// Returns the number of points written (or a negative error).
int64_t orc_points(int64_t n, const uint8_t* etype, const double* verts, const double* sigma, int level, double* xyzq) {
    if (level < 0 || level > 4) return ERR_BAD_RULE;
    int64_t c = 0;
    std::vector<Pt<long double>> p;
    for (int64_t e = 0; e < n; ++e) {
        Geom<long double> g;
        int rc = make_geom<long double>(etype[e], verts + 9 * e, g);
        if (rc) return rc;
        element_points<long double>(g, level, p);
        for (auto& q : p) {
            if (xyzq) { xyzq[4 * c] = (double)q.x; xyzq[4 * c + 1] = (double)q.y; xyzq[4 * c + 2] = (double)q.z; xyzq[4 * c + 3] = (double)(q.w * (long double)sigma[e] * g.area); }
            ++c;
        }
    }
    return c;
}

// Default DR limits dr[2][5] ([0] = triangle, [1] = rectangle; entries = upper limits of
// {analytic, N=33, N=19|17, N=12, N=7}).  want_field = 0: the printed triangle-potential
// limits 3/8/20/80/1500 (L159), used for both element types (rectangle limits are not
// printed); want_field = 1: limits for Phi and E together ("slightly higher", L159; values
// re-derived with the paper's protocol, DESIGN.md §3 reading 7).
int orc_default_policy(double* dr, int want_field) {
    static const double pot[5] = {3, 8, 20, 80, 1500};
    static const double ftri[5] = {4, 10, 25, 100, 2000};
    static const double frect[5] = {6, 15, 40, 150, 3000};
    // want_field = 2: limits for single-precision evaluation - the distance ratio from which each
    // rule's own field error is below the FP32 rounding floor of 1e-7 (same protocol, reading 7)
    static const double f32tri[5] = {2, 2, 3, 6, 25};
    static const double f32rect[5] = {2, 3, 4, 8, 30};
    if (want_field < 0 || want_field > 2) return ERR_INVALID;
    for (int b = 0; b < 5; ++b) {
        dr[b] = want_field == 2 ? f32tri[b] : want_field ? ftri[b] : pot[b];
        dr[5 + b] = want_field == 2 ? f32rect[b] : want_field ? frect[b] : pot[b];
    }
    return ERR_OK;
}

int orc_choose_level(double D2, double L, const double* dr5, int levels_mask) { return choose_level(D2, L, dr5, levels_mask); }

// precision: 0 = long double (parity), 1 = double (timed CPU baseline).  level -1 = adaptive.
// npi[m] / nana[m] (may be null): point-charge interactions / analytic pairs used per field point.
int orc_eval(int64_t n, const uint8_t* etype, const double* verts, const double* sigma, int level,
             const double* dr, int levels_mask, int64_t m, const double* pts, double* phi, double* E,
             double* Sphi, double* SE, int64_t* npi, int64_t* nana, int precision, int nthreads) {
    if (precision == 0)
        return eval_impl<long double>(n, etype, verts, sigma, level, dr, levels_mask, m, pts, phi, E, Sphi, SE, npi, nana, nthreads);
    return eval_impl<double>(n, etype, verts, sigma, level, dr, levels_mask, m, pts, phi, E, Sphi, SE, npi, nana, nthreads);
}

// Linear sigma over each element (L275), long double, cubature levels only.
int orc_eval_linear(int64_t n, const uint8_t* etype, const double* verts, const double* sigma_v, int level,
                    const double* dr, int levels_mask, int64_t m, const double* pts, double* phi, double* E,
                    double* Sphi, double* SE) {
    return linear_impl<long double>(n, etype, verts, sigma_v, level, dr, levels_mask, m, pts, phi, E, Sphi, SE);
}

// Field gradient (L273), long double, cubature levels only.
int orc_eval_gradient(int64_t n, const uint8_t* etype, const double* verts, const double* sigma, int level,
                      const double* dr, int levels_mask, int64_t m, const double* pts, double* G, double* SG) {
    return grad_impl<long double>(n, etype, verts, sigma, level, dr, levels_mask, m, pts, G, SG);
}

// Unit-sigma integrals of Eq. 2.1 without the 1/(4 pi eps0) prefactor, three ways.
int orc_analytic(int etype, const double* verts9, const double* P, double* Iphi, double* IE, int precision) {
    if (precision == 0) {
        Geom<long double> g;
        int rc = make_geom<long double>(etype, verts9, g);
        if (rc) return rc;
        long double ip; V3<long double> ie;
        analytic_integrals<long double>(g, {(long double)P[0], (long double)P[1], (long double)P[2]}, ip, ie);
        *Iphi = (double)ip; IE[0] = (double)ie.x; IE[1] = (double)ie.y; IE[2] = (double)ie.z;
    } else {
        Geom<double> g;
        int rc = make_geom<double>(etype, verts9, g);
        if (rc) return rc;
        double ip; V3<double> ie;
        analytic_integrals<double>(g, {P[0], P[1], P[2]}, ip, ie);
        *Iphi = ip; IE[0] = ie.x; IE[1] = ie.y; IE[2] = ie.z;
    }
    return ERR_OK;
}

int orc_gl2(int etype, const double* verts9, const double* P, int ngl, double* Iphi, double* IE) {
    Geom<long double> g;
    int rc = make_geom<long double>(etype, verts9, g);
    if (rc) return rc;
    F4 r;
    gl2_integrals(g, {(long double)P[0], (long double)P[1], (long double)P[2]}, ngl, r);
    *Iphi = (double)r.v[0]; IE[0] = (double)r.v[1]; IE[1] = (double)r.v[2]; IE[2] = (double)r.v[3];
    return ERR_OK;
}

int orc_adaptive(int etype, const double* verts9, const double* P, double reltol, double* Iphi, double* IE, double* errest) {
    Geom<long double> g;
    int rc = make_geom<long double>(etype, verts9, g);
    if (rc) return rc;
    Adaptive a(g, {(long double)P[0], (long double)P[1], (long double)P[2]}, (long double)reltol);
    F4 r = a.run();
    *Iphi = (double)r.v[0]; IE[0] = (double)r.v[1]; IE[1] = (double)r.v[2]; IE[2] = (double)r.v[3];
    if (errest) *errest = (double)a.err;
    return ERR_OK;
}

int orc_gauss_legendre(int n, double* x, double* w) {
    std::vector<long double> xx, ww;
    gauss_legendre(n, xx, ww);
    for (int i = 0; i < n; ++i) { x[i] = (double)xx[i]; w[i] = (double)ww[i]; }
    return ERR_OK;
}

// Collocation-matrix rows (L34): A_ij = k * Int_{elem j} dS / |c_i - Q| with unit sigma,
// c_i = centroid of element i; per pair the rule by DR(i,j) (L159), analytic below the first
// limit (self term included: D = 0).  code[r][j] = level used (0..4) or 5 = analytic.
int orc_assemble_rows(int64_t n, const uint8_t* etype, const double* verts, const double* dr, int levels_mask,
                      int64_t nrows, const int64_t* rows, double* out, uint8_t* code, int precision, int nthreads) {
    typedef long double T;
    (void)precision;
    std::vector<Geom<T>> G(n);
    for (int64_t e = 0; e < n; ++e) {
        int rc = make_geom<T>(etype[e], verts + 9 * e, G[e]);
        if (rc) return rc;
    }
    const T k = coulomb_k();
    const int nt = threads_for(nthreads);
#pragma omp parallel for schedule(dynamic, 1) num_threads(nt)
    for (int64_t r = 0; r < nrows; ++r) {
        const int64_t i = rows[r];
        const V3<T> P = G[i].cen;
        const double px = (double)P.x, py = (double)P.y, pz = (double)P.z;
        std::vector<Pt<T>> p;
        for (int64_t j = 0; j < n; ++j) {
            const Geom<T>& g = G[j];
            double dx = px - (double)g.cen.x, dy = py - (double)g.cen.y, dz = pz - (double)g.cen.z;
            int lv = choose_level(dx * dx + dy * dy + dz * dz, (double)g.L, dr + 5 * g.type, levels_mask);
            T val = 0;
            if (lv == 5) {
                T ip; V3<T> ie;
                analytic_integrals<T>(g, P, ip, ie);
                val = ip;
            } else {
                element_points<T>(g, lv, p);
                for (const Pt<T>& q : p) {
                    const T ddx = P.x - q.x, ddy = P.y - q.y, ddz = P.z - q.z;
                    val += q.w * g.area / sqrtl(ddx * ddx + ddy * ddy + ddz * ddz);
                }
            }
            out[r * n + j] = (double)(k * val);
            if (code) code[r * n + j] = (uint8_t)lv;
        }
    }
    return ERR_OK;
}

// Element k seen from field point k (no sum): see pairs_impl.  precision 0 = long double, 1 = double.
int orc_eval_pairs(int64_t K, const uint8_t* etype, const double* verts, const double* sigma, int method,
                   const double* dr, int levels_mask, const double* pts, double* phi, double* E, double* Sphi,
                   double* SE, uint8_t* used, int precision) {
    if (precision == 0) return pairs_impl<long double>(K, etype, verts, sigma, method, dr, levels_mask, pts, phi, E, Sphi, SE, used);
    return pairs_impl<double>(K, etype, verts, sigma, method, dr, levels_mask, pts, phi, E, Sphi, SE, used);
}

// Duffy-mapped rectangle rule of `level` on the reference triangle A=(0,0), B=(1,0), C=(0,1):
// bary[N][3] = (lambda_A, lambda_B, lambda_C) of each node, w[N] = its weight relative to the area.
int orc_duffy_nodes(int level, double* bary, double* w) {
    if (level < 0 || level > 4) return ERR_BAD_RULE;
    const double ref[9] = {0, 0, 0, 1, 0, 0, 0, 1, 0};
    Geom<long double> g;
    make_geom<long double>(TRI, ref, g);
    std::vector<Pt<long double>> p;
    element_points_duffy<long double>(g, level, p);
    for (size_t i = 0; i < p.size(); ++i) {
        bary[3 * i] = (double)(1 - p[i].x - p[i].y); bary[3 * i + 1] = (double)p[i].x; bary[3 * i + 2] = (double)p[i].y;
        w[i] = (double)p[i].w;
    }
    return ERR_OK;
}

// sum_i w'_i x_i^a y_i^b - a! b! 2/(a+b+2)!  for the Duffy-mapped rule on the reference triangle (long double).
double orc_duffy_monomial_residual(int level, int a, int b) {
    const double ref[9] = {0, 0, 0, 1, 0, 0, 0, 1, 0};
    Geom<long double> g;
    make_geom<long double>(TRI, ref, g);
    std::vector<Pt<long double>> p;
    element_points_duffy<long double>(g, level, p);
    long double s = 0;
    for (auto& q : p) s += q.w * powl(q.x, a) * powl(q.y, b);
    long double num = 2, den = 1;
    for (int i = 2; i <= a; ++i) num *= i;
    for (int i = 2; i <= b; ++i) num *= i;
    for (int i = 2; i <= a + b + 2; ++i) den *= i;
    return (double)(s - num / den);
}

int orc_num_threads() {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

}  // extern "C"
