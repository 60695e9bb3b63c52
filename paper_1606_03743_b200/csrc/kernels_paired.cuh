// Steps a2 + a3 + a4 for meshes with rectangles: the evaluation kernel with the rectangle rules'
// points taken in SYMMETRIC PAIRS.
//
// Every rectangle rule of App. B consists of point pairs (x, y), (-x, -y) of equal
// weight, plus the centre in the 7-, 17- and 33-point rules.  By Eq. 3.2 (L103) the two points of a pair
// sit at Q = C +- d on the element (C the centre, d = (a/2) x u_x + (b/2) y u_y), so with D = P - C
//     |P - Q|^2 = (|D|^2 + |d|^2) -+ 2 D.d ,
// and D, |D|^2 are shared by all points of the element, D.d by the two points of a pair.  The pair's
// contribution to Eq. 4.1 (L139-143) is then
//     Phi += q (y+ + y-),    E += q (y+^3 + y-^3) D + (y-^3 - y+^3) (q d) ,    y = 1/|P - Q| ,
// with the first E term summed per element (S = sum of q y^3, one multiply-add with D at the end) and
// q d stored beside d.  That is 28 FP64 instructions per pair instead of 36, and 9 instead of 18 for the
// centre point: 102 instead of 126 per 7-point element, 177 instead of 216 per 12-point element (bare
// loops on B200 with 30 per pair: 1.08e12 against 0.93e12 point-charge interactions/s).
// The sums are the sums of Eq. 4.1 term by term;
// only the rounding differs (|D|^2 + |d|^2 -+ 2 D.d loses nothing as long as |d| < |D|, i.e. at every
// distance ratio a cubature rule is used at; the host takes this kernel only under policies whose
// analytic limit for rectangles is >= 2).  Triangle rules have no central symmetry; the 7-point one has its
// points on the medians and is taken in a similar form (consume_tri7 below); the other triangle rules, and
// all elements in the pair-by-pair and analytic branches, go through the same code as in eval_adaptive_kernel.
//
// Potential-only calls (out_E = NULL: the mat-vec of a BEM solve, L34) take the same forms without their field
// part: 18 instead of 24 FP64 instructions per pair, 6 instead of 12 for a centre point.
//
// Same execution model as kernels_eval.cuh (persistent CTAs, autonomous warps, atomic work queue, per-warp
// double-buffered bulk-TMA windows).  A stage of the window holds whole elements in batch order; a small
// run table beside it says which stretches are paired rectangles of one level (element blocks: centre
// record + pair records) and which are plain point records.
#pragma once
#include "kernels_eval.cuh"

namespace bemcub {

// pair tables, filled by bemcub_create from rules.h: per level the pairs' plus members (x, y, w, 0), the
// weight of the centre point (0 if the rule has none) and the number of pairs (0: level not pairable)
__constant__ double c_pair_tab[5 * 16 * 4];
__constant__ double c_pair_center_w[5];
__constant__ int c_pair_np[5];

// Element block of a paired rectangle, in 32-byte units of the window:
//   [C.x C.y C.z q_centre] [d.x d.y d.z q | |d|^2 q d.x q d.y q d.z] x NP      = 1 + 2 NP units
__host__ __device__ constexpr int pair_units(int np) { return 1 + 2 * np; }

// One thread per (element, slot): slot 0 writes the centre record, slot k > 0 pair k - 1.  Triangles are skipped.
__global__ void expand_pairs_kernel(int64_t n, int level, int np, const uint8_t* __restrict__ type, const double* __restrict__ verts,
                                    const double4* __restrict__ cenL, const double* __restrict__ area,
                                    const double* __restrict__ sigma, double* __restrict__ out) {
  const int64_t idx = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (idx >= n * (np + 1)) return;
  const int64_t e = idx / (np + 1);
  const int slot = (int)(idx - e * (np + 1));
  if (type[e] != 1) return;
  const double* v = verts + 9 * e;
  const double q = (sigma ? sigma[e] : 1.0) * area[e];  // q = sigma A (L143)
  double* blk = out + e * (int64_t)(4 * pair_units(np));
  if (slot == 0) {
    const double4 c = cenL[e];
    blk[0] = c.x; blk[1] = c.y; blk[2] = c.z; blk[3] = c_pair_center_w[level] * q;
  } else {
    const double* r = c_pair_tab + 4 * (16 * level + slot - 1);
    const double xs = 0.5 * r[0], ys = 0.5 * r[1];
    // Eq. 3.2: Q - Q_cen = (a/2) x u_x + (b/2) y u_y, with a u_x = P1 - P0 and b u_y = P3 - P0
    const double dx = fma(ys, v[6] - v[0], xs * (v[3] - v[0]));
    const double dy = fma(ys, v[7] - v[1], xs * (v[4] - v[1]));
    const double dz = fma(ys, v[8] - v[2], xs * (v[5] - v[2]));
    double* p = blk + 4 + 8 * (slot - 1);
    const double qk = r[2] * q;
    p[0] = dx; p[1] = dy; p[2] = dz; p[3] = qk;
    p[4] = fma(dx, dx, fma(dy, dy, dz * dz)); p[5] = qk * dx; p[6] = qk * dy; p[7] = qk * dz;
  }
}

// `nelem` element blocks of NP pairs (+ centre if HC) applied to the lane's R field points.
// MODE = kModePhi (potential only: the mat-vec of a BEM solve, any call without out_E): 18 per pair, 6 for the centre.
template <int R, int NP, bool HC, int MODE>
__device__ __forceinline__ void consume_pairs(const double4* __restrict__ buf, int nelem, const double (&px)[R], const double (&py)[R],
                                              const double (&pz)[R], Accum<double, R, MODE>& a) {
  constexpr bool kE = MODE != kModePhi;
  constexpr int UNITS = pair_units(NP);
  const double c375 = c_three_eighths;
#pragma unroll 1
  for (int e = 0; e < nelem; ++e) {
    const double4* blk = buf + e * UNITS;
    const double4 c = blk[0];
    double Dx[R], Dy[R], Dz[R], D2[R], S[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
      Dx[r] = __dsub_rn(px[r], c.x); Dy[r] = __dsub_rn(py[r], c.y); Dz[r] = __dsub_rn(pz[r], c.z);
      const double yz = __fma_rn(Dy[r], Dy[r], __dmul_rn(Dz[r], Dz[r]));
      D2[r] = __fma_rn(Dx[r], Dx[r], yz);
      S[r] = 0.0;
      if constexpr (HC) {  // the centre point: |P - Q| = |D|
        const double y = rsqrt_f64(D2[r], yz, c375);
        a.phi[r] = __fma_rn(c.w, y, a.phi[r]);
        if constexpr (kE) S[r] = __dmul_rn(c.w, __dmul_rn(y, __dmul_rn(y, y)));
      }
    }
    constexpr int kUnroll = NP <= 3 ? NP : 1;  // (partial unrolling of the longer rules: no difference measured)
#pragma unroll kUnroll
    for (int k = 0; k < NP; ++k) {
      const double4 a0 = blk[1 + 2 * k], a1 = blk[2 + 2 * k];  // d, q | |d|^2, q d
#pragma unroll
      for (int r = 0; r < R; ++r) {
        const double B = __fma_rn(Dx[r], a0.x, __fma_rn(Dy[r], a0.y, __dmul_rn(Dz[r], a0.z)));  // D.d
        const double A = __dadd_rn(D2[r], a1.x);
        const double rp = __fma_rn(-2.0, B, A), rm = __fma_rn(2.0, B, A);  // |P - (C + d)|^2, |P - (C - d)|^2
        const double yp = rsqrt_f64(rp, A, c375), ym = rsqrt_f64(rm, B, c375);
        a.phi[r] = __fma_rn(a0.w, __dadd_rn(yp, ym), a.phi[r]);
        if constexpr (kE) {
          const double cp = __dmul_rn(yp, __dmul_rn(yp, yp)), cm = __dmul_rn(ym, __dmul_rn(ym, ym));
          // E += q y+^3 (D - d) + q y-^3 (D + d) = q (y+^3 + y-^3) D + (y-^3 - y+^3) (q d)
          S[r] = __fma_rn(a0.w, __dadd_rn(cp, cm), S[r]);
          const double t = __dsub_rn(cm, cp);
          a.ex[r] = __fma_rn(t, a1.y, a.ex[r]);
          a.ey[r] = __fma_rn(t, a1.z, a.ey[r]);
          a.ez[r] = __fma_rn(t, a1.w, a.ez[r]);
        }
      }
    }
    if constexpr (kE) {
#pragma unroll
      for (int r = 0; r < R; ++r) {
        a.ex[r] = __fma_rn(S[r], Dx[r], a.ex[r]);
        a.ey[r] = __fma_rn(S[r], Dy[r], a.ey[r]);
        a.ez[r] = __fma_rn(S[r], Dz[r], a.ez[r]);
      }
    }
  }
}

// ------------------------------------------------------------------------------------------------
// The 7-point triangle rule (Table A2) the same way.  Its points are the centroid and two
// orbits (a, b, b) over the three vertices, and by Eq. 3.3 a point with the large weight on vertex V is
//     Q = a V + b (the other two) = C + kappa (V - C),   kappa = a - b,
// so the six points sit on the three medians: with u_V = V - C and D = P - C,
//     |P - Q|^2 = (|D|^2 + kappa^2 |u_V|^2) - 2 kappa D.u_V ,
// D.u_V is shared by the two points of a median, D and |D|^2 by all seven points, and
//     E += q y^3 (D - kappa u_V) = (q y^3) D + y^3 (-q kappa u_V)
// with the first term summed per element.  14 FP64 instructions per point, 111 instead of 126 per element.
__constant__ double c_tri7_kappa[2];  // kappa of the two orbits (0, 0: the table does not have this structure)
__constant__ double c_tri7_w[3];      // weights: centroid, orbit 1, orbit 2
constexpr int kTri7Units = 16;        // [C, q0] + 3 x ([u_V, 0] + 2 x ([-2 kappa, kappa^2 |u|^2, q, 0] [-q kappa u_V, 0]))
constexpr int kClsTri7 = 6;

// One thread per (element, slot): slot 0 the centroid record, slot 1..3 the records of one median.  Rectangles are skipped.
__global__ void expand_tri7_kernel(int64_t n, const uint8_t* __restrict__ type, const double* __restrict__ verts,
                                   const double4* __restrict__ cenL, const double* __restrict__ area,
                                   const double* __restrict__ sigma, double* __restrict__ out) {
  const int64_t idx = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (idx >= 4 * n) return;
  const int64_t e = idx >> 2;
  const int slot = (int)(idx & 3);
  if (type[e] != 0) return;
  const double q = (sigma ? sigma[e] : 1.0) * area[e];  // q = sigma A (L143)
  const double4 c = cenL[e];
  double* blk = out + e * (int64_t)(4 * kTri7Units);
  if (slot == 0) {
    blk[0] = c.x; blk[1] = c.y; blk[2] = c.z; blk[3] = c_tri7_w[0] * q;
    return;
  }
  const double* v = verts + 9 * e + 3 * (slot - 1);
  const double ux = v[0] - c.x, uy = v[1] - c.y, uz = v[2] - c.z;
  const double u2 = fma(ux, ux, fma(uy, uy, uz * uz));
  double* p = blk + 4 + 20 * (slot - 1);
  p[0] = ux; p[1] = uy; p[2] = uz; p[3] = 0.0;
#pragma unroll
  for (int o = 0; o < 2; ++o) {
    const double k = c_tri7_kappa[o], qo = c_tri7_w[1 + o] * q;
    double* r = p + 4 + 8 * o;
    r[0] = -2.0 * k; r[1] = k * k * u2; r[2] = qo; r[3] = 0.0;
    r[4] = -qo * k * ux; r[5] = -qo * k * uy; r[6] = -qo * k * uz; r[7] = 0.0;
  }
}

template <int R, int MODE>
__device__ __forceinline__ void consume_tri7(const double4* __restrict__ buf, int nelem, const double (&px)[R], const double (&py)[R],
                                             const double (&pz)[R], Accum<double, R, MODE>& a) {
  constexpr bool kE = MODE != kModePhi;
  const double c375 = c_three_eighths;
#pragma unroll 1
  for (int e = 0; e < nelem; ++e) {
    const double4* blk = buf + e * kTri7Units;
    const double4 c = blk[0];
    double Dx[R], Dy[R], Dz[R], D2[R], S[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
      Dx[r] = __dsub_rn(px[r], c.x); Dy[r] = __dsub_rn(py[r], c.y); Dz[r] = __dsub_rn(pz[r], c.z);
      const double yz = __fma_rn(Dy[r], Dy[r], __dmul_rn(Dz[r], Dz[r]));
      D2[r] = __fma_rn(Dx[r], Dx[r], yz);
      const double y = rsqrt_f64(D2[r], yz, c375);  // the centroid point
      a.phi[r] = __fma_rn(c.w, y, a.phi[r]);
      S[r] = kE ? __dmul_rn(c.w, __dmul_rn(y, __dmul_rn(y, y))) : 0.0;
    }
#pragma unroll
    for (int i = 0; i < 3; ++i) {
      const double4 u = blk[1 + 5 * i];
      double B[R];
#pragma unroll
      for (int r = 0; r < R; ++r) B[r] = __fma_rn(Dx[r], u.x, __fma_rn(Dy[r], u.y, __dmul_rn(Dz[r], u.z)));  // D.u_V
#pragma unroll
      for (int o = 0; o < 2; ++o) {
        const double4 p0 = blk[2 + 5 * i + 2 * o], p1 = blk[3 + 5 * i + 2 * o];  // -2 kappa, kappa^2 |u|^2, q | -q kappa u
#pragma unroll
        for (int r = 0; r < R; ++r) {
          const double A = __dadd_rn(D2[r], p0.y);
          const double r2 = __fma_rn(p0.x, B[r], A);
          const double y = rsqrt_f64(r2, A, c375);
          a.phi[r] = __fma_rn(p0.z, y, a.phi[r]);
          if constexpr (kE) {
            const double y3 = __dmul_rn(y, __dmul_rn(y, y));
            S[r] = __fma_rn(p0.z, y3, S[r]);
            a.ex[r] = __fma_rn(y3, p1.x, a.ex[r]);
            a.ey[r] = __fma_rn(y3, p1.y, a.ey[r]);
            a.ez[r] = __fma_rn(y3, p1.z, a.ez[r]);
          }
        }
      }
    }
    if constexpr (kE) {
#pragma unroll
      for (int r = 0; r < R; ++r) {
        a.ex[r] = __fma_rn(S[r], Dx[r], a.ex[r]);
        a.ey[r] = __fma_rn(S[r], Dy[r], a.ey[r]);
        a.ez[r] = __fma_rn(S[r], Dz[r], a.ez[r]);
      }
    }
  }
}

struct PairedParams {
  AdaptiveParams ad;           // everything eval_adaptive_kernel takes (lvl_pts: the plain point records of every level)
  const double4* pair_pts[5];  // element blocks of the rectangles per level (n * pair_units(np) units; triangles' blocks unused)
  int pair_np[5];              // pairs per level, 0 = this level's rectangles are streamed as plain points
  const double4* tri7_pts;     // element blocks of the triangles for the 7-point rule (n * kTri7Units units), or null
};

// per-warp bookkeeping in shared memory: the adaptive kernel's, plus the run table of each stage
struct PairedScratch {
  WarpScratch s;
  unsigned long long n_saved;  // FP64 instructions per field point the paired form did NOT execute (against 18 per interaction)
  uint32_t run[kStages][32];  // class (0..4: paired rectangles of that level, 5: point records, 6: 7-point triangles) | offset << 3 | length << 11, in units
};
constexpr int kClsPoints = 5;

template <int WARPS>
constexpr size_t paired_smem_bytes() {
  return (size_t)WARPS * (kStages * kBuf * sizeof(double4) + kStages * 8 + sizeof(PairedScratch));
}

template <int R, int WARPS, int MODE = kModePhiE>
__global__ void __launch_bounds__(WARPS * 32, 1) eval_paired_kernel(const __grid_constant__ PairedParams pp) {
  static_assert(MODE == kModePhiE || MODE == kModePhi, "Phi + E or Phi only");
  typedef double4 P4;
  const AdaptiveParams& p = pp.ad;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  P4* const win = reinterpret_cast<P4*>(smem_raw) + (size_t)warp * kStages * kBuf;
  unsigned char* const after_win = smem_raw + (size_t)WARPS * kStages * kBuf * sizeof(P4);
  const uint32_t bar0 = smem_u32(reinterpret_cast<uint64_t*>(after_win) + warp * kStages);
  PairedScratch* const ps = reinterpret_cast<PairedScratch*>(after_win + (size_t)WARPS * kStages * 8) + warp;
  WarpScratch* const scr = &ps->s;
  const uint32_t win0 = smem_u32(win);
  if (lane == 0) {
    mbar_init(bar0, 1);
    mbar_init(bar0 + 8, 1);
    mbar_fence_init();
    scr->n_inter = 0;
    scr->n_ana = 0;
    ps->n_saved = 0;
  }
  __syncwarp();
  uint32_t phases = 0;
  const unsigned lt_mask = (1u << lane) - 1u;
  KernelClock clk;
  clk.begin();

  for (;;) {
    const int64_t item = next_item(p.queue, lane);
    if (item >= p.nitems) break;
    const int64_t split = item / p.ntiles, tile = item - split * p.ntiles;

    WarpTile<R> w;
    w.first = tile * (32 * R);
    w.m = p.m;
    load_field_points<double, R>(p.field, p.m, tile, lane, w.px, w.py, w.pz);
    {  // bounding sphere of the tile, non-finite points left out (see eval_adaptive_kernel)
      const double nan = CUDART_NAN;
      double lox = nan, hix = nan, loy = nan, hiy = nan, loz = nan, hiz = nan;
      int cntok = 0;
#pragma unroll
      for (int r = 0; r < R; ++r) {
        cntok += w.ok(r, lane) ? 1 : 0;
        const bool fin = isfinite(w.px[r]) && isfinite(w.py[r]) && isfinite(w.pz[r]);
        const double bx = fin ? w.px[r] : nan, by = fin ? w.py[r] : nan, bz = fin ? w.pz[r] : nan;
        lox = fmin(lox, bx); hix = fmax(hix, bx);
        loy = fmin(loy, by); hiy = fmax(hiy, by);
        loz = fmin(loz, bz); hiz = fmax(hiz, bz);
      }
      lox = warp_min(lox); hix = warp_max(hix);
      loy = warp_min(loy); hiy = warp_max(hiy);
      loz = warp_min(loz); hiz = warp_max(hiz);
      const bool any_fin = lox <= hix;
      const double cx = any_fin ? 0.5 * (lox + hix) : 0.0, cy = any_fin ? 0.5 * (loy + hiy) : 0.0,
                   cz = any_fin ? 0.5 * (loz + hiz) : 0.0;
      double d2 = 0.0;
#pragma unroll
      for (int r = 0; r < R; ++r) {
        const double dx = w.px[r] - cx, dy = w.py[r] - cy, dz = w.pz[r] - cz;
        const double t = dx * dx + dy * dy + dz * dz;
        d2 = fmax(d2, t <= 1e300 ? t : 0.0);
      }
      const double rho = sqrt(warp_max(d2));
      cntok = warp_sum(cntok);
      __syncwarp();
      if (lane == 0) {
        scr->cx = cx; scr->cy = cy; scr->cz = cz; scr->rho = rho;
        scr->mag = fmax(fmax(fabs(cx), fabs(cy)), fabs(cz)) + rho;
        scr->nvalid = cntok;
      }
      __syncwarp();
    }

    const int64_t e_begin = split * p.elems_per_split;
    const int64_t e_end = min(p.n, e_begin + p.elems_per_split);
    Accum<double, R, MODE> tot;
    tot.zero();

    // state of the current 32-element batch: lane l holds element batch0 + l
    int64_t batch_next = e_begin;
    int cnt = 0, pre = 0, total = 0, cls = kClsPoints, key = -1, estride = 0, realn = 0, saved = 0, cursor = 32;
    const P4* src = nullptr;

    // Fills `stage` with the next round of whole elements; returns the number of runs (0 = done).
    auto produce = [&](int stage) -> int {
      for (;;) {
        if (cursor < 32) {
          const int first = cursor;
          const int base = __shfl_sync(kFullMask, pre, first);
          const bool after = lane >= first;
          const unsigned nofit = __ballot_sync(kFullMask, after && (pre + cnt - base > kBuf));
          const int next = nofit ? (__ffs(nofit) - 1) : 32;
          const int pre_next = __shfl_sync(kFullMask, pre, next & 31);
          const int endp = (next < 32) ? pre_next : total;
          const int nstage = endp - base;
          cursor = next;
          if (nstage == 0) continue;
          const bool inc = after && lane < next && cnt > 0;
          const unsigned incmask = __ballot_sync(kFullMask, inc);
          // copies: consecutive elements of one array whose blocks are adjacent in memory share one
          const int prev_cnt = __shfl_up_sync(kFullMask, cnt, 1), prev_key = __shfl_up_sync(kFullMask, key, 1);
          const bool cont = inc && lane > first && prev_cnt > 0 && prev_key == key && prev_cnt == estride;
          const unsigned heads = __ballot_sync(kFullMask, inc && !cont);
          const unsigned higher = heads & ~((2u << lane) - 1u);
          const int h2 = higher ? (__ffs(higher) - 1) : 32;
          const int pre_h2 = __shfl_sync(kFullMask, pre, h2 & 31);
          const int copy_end = (h2 < 32) ? pre_h2 : endp;
          // runs: maximal stretches of streamed elements of one class (elements that are not streamed do not break one)
          const unsigned below = incmask & lt_mask;
          const int pl = below ? (31 - __clz(below)) : -1;
          const int prev_cls = __shfl_sync(kFullMask, cls, pl & 31);
          const bool rhead = inc && (pl < 0 || prev_cls != cls);
          const unsigned rheads = __ballot_sync(kFullMask, rhead);
          const unsigned rhigher = rheads & ~((2u << lane) - 1u);
          const int r2 = rhigher ? (__ffs(rhigher) - 1) : 32;
          const int pre_r2 = __shfl_sync(kFullMask, pre, r2 & 31);
          const int run_end = (r2 < 32) ? pre_r2 : endp;
          if (rhead) ps->run[stage][__popc(rheads & lt_mask)] = (uint32_t)cls | ((uint32_t)(pre - base) << 3) | ((uint32_t)(run_end - pre) << 11);
          const int nreal = warp_sum(inc ? realn : 0), nsaved = warp_sum(inc ? saved : 0);
          if (lane == 0) {
            mbar_arrive_expect_tx(bar0 + 8 * stage, (uint32_t)(nstage * sizeof(P4)));
            scr->n_inter += (unsigned long long)nreal * scr->nvalid;
            ps->n_saved += (unsigned long long)nsaved * scr->nvalid;
          }
          __syncwarp();
          if (inc && !cont)
            tma_load_1d(win0 + (uint32_t)((stage * kBuf + (pre - base)) * sizeof(P4)), src, (uint32_t)((copy_end - pre) * sizeof(P4)),
                        bar0 + 8 * stage);
          return __popc(rheads);
        }
        if (batch_next >= e_end) return 0;
        // ---- a2: classify 32 elements, one per lane, against the tile's bounding sphere
        const int64_t batch0 = batch_next;
        const int64_t e = batch0 + lane;
        batch_next += 32;
        cnt = 0;
        realn = 0;
        saved = 0;
        key = -1;
        cls = kClsPoints;
        bool is_ana = false, is_mixed = false;
        if (e < e_end) {
          const double4 c = p.cenL[e];
          const int t = p.type[e];
          const double rho = scr->rho;
          const double dx = scr->cx - c.x, dy = scr->cy - c.y, dz = scr->cz - c.z;
          const double Dc = sqrt(dx * dx + dy * dy + dz * dz);
          const double slack = 1e-9 * (Dc + rho) + 1e-12 * (scr->mag + fmax(fmax(fabs(c.x), fabs(c.y)), fabs(c.z)));
          const double Dhi = Dc + rho + slack;
          const double Dlo = fmax(Dc - rho - slack, 0.0);
          const int lfar = p.pol.map[want_level(Dhi * Dhi, c.w, p.pol.dr[t])];
          const int lnear = p.pol.map[want_level(Dlo * Dlo, c.w, p.pol.dr[t])];
          if (lnear != lfar && (!p.pol.allow_upgrade || lnear == 5)) {
            is_mixed = true;
          } else if (lnear == 5) {
            is_ana = true;
          } else {
            const int lvl = lnear;
            realn = rule_npts(t, lvl);
            const int np = (t == 1) ? pp.pair_np[lvl] : 0;
            if (np > 0) {  // a rectangle in paired form
              cls = lvl;
              key = lvl;
              cnt = estride = pair_units(np);
              src = pp.pair_pts[lvl] + e * estride;
              // 9 per element (D, |D|^2, S D), 9 for a centre point, 28 per pair - instead of 18 per point
              // (Phi only: 6, 6 and 18 instead of 12 per point)
              saved = MODE == kModePhi ? 12 * realn - (6 + (realn > 2 * np ? 6 : 0) + 18 * np)
                                       : 18 * realn - (9 + (realn > 2 * np ? 9 : 0) + 28 * np);
            } else if (t == 0 && lvl == 1 && pp.tri7_pts) {  // a triangle with the 7-point rule in median form
              cls = kClsTri7;
              key = 16;
              cnt = estride = kTri7Units;
              src = pp.tri7_pts + e * kTri7Units;
              saved = MODE == kModePhi ? 12 * 7 - 69 : 18 * 7 - 111;
            } else {
              key = 8 + lvl;
              cnt = realn;
              estride = p.stride[lvl];
              src = reinterpret_cast<const P4*>(p.lvl_pts[lvl]) + e * p.stride[lvl];
            }
          }
        }
        pre = warp_excl_scan(cnt, lane, &total);
        cursor = 0;
        unsigned amask = __ballot_sync(kFullMask, is_ana), xmask = __ballot_sync(kFullMask, is_mixed);
        if (amask) {
          bool all_ok[R];
#pragma unroll
          for (int r = 0; r < R; ++r) all_ok[r] = w.ok(r, lane);
          if (lane == 0) scr->n_ana += (unsigned long long)__popc(amask) * scr->nvalid;
          while (amask) {
            const int l = __ffs(amask) - 1;
            amask &= amask - 1;
            analytic_element<R, MODE>(p, batch0 + l, w, all_ok, tot);
          }
        }
        while (xmask) {
          const int l = __ffs(xmask) - 1;
          xmask &= xmask - 1;
          mixed_element<double, R, MODE>(p, batch0 + l, w, w.px, w.py, w.pz, lane, tot, scr);
        }
      }
    };

    // all runs of a filled stage applied to the warp's field points
    auto consume_stage = [&](int stage, int nruns) {
      for (int k = 0; k < nruns; ++k) {
        const uint32_t ent = ps->run[stage][k];
        const P4* b = win + stage * kBuf + ((ent >> 3) & 255u);
        const int len = (int)(ent >> 11);
        switch (ent & 7u) {
          case 0: consume_pairs<R, 2, false, MODE>(b, len / pair_units(2), w.px, w.py, w.pz, tot); break;
          case 1: consume_pairs<R, 3, true, MODE>(b, len / pair_units(3), w.px, w.py, w.pz, tot); break;
          case 2: consume_pairs<R, 6, false, MODE>(b, len / pair_units(6), w.px, w.py, w.pz, tot); break;
          case 3: consume_pairs<R, 8, true, MODE>(b, len / pair_units(8), w.px, w.py, w.pz, tot); break;
          case 4: consume_pairs<R, 16, true, MODE>(b, len / pair_units(16), w.px, w.py, w.pz, tot); break;
          case kClsTri7: consume_tri7<R, MODE>(b, len / kTri7Units, w.px, w.py, w.pz, tot); break;
          default: consume_into<R, MODE>(b, len, w.px, w.py, w.pz, tot); break;
        }
      }
    };

    // software pipeline with a single produce() call site: fill stage s^1, then consume stage s
    int cur = 0, stage = 1;
    for (;;) {
      const int nxt = produce(stage ^ 1);
      if (cur > 0) {
        mbar_wait(bar0 + 8 * stage, (phases >> stage) & 1u);
        phases ^= 1u << stage;
        consume_stage(stage, cur);
        __syncwarp();
      }
      if (nxt == 0) break;
      stage ^= 1;
      cur = nxt;
    }
    store_partial<R, MODE>(p.partial + split * p.split_stride, nullptr, p.m, tile, lane, tot);
  }

  __syncwarp();
  if (p.counters && lane == 0) {
    if (scr->n_inter) atomicAdd(p.counters, scr->n_inter);
    if (scr->n_ana) atomicAdd(p.counters + 1, scr->n_ana);
    if (ps->n_saved) atomicAdd(p.counters + 3, ps->n_saved);
  }
  clk.end(p.counters);
}

}  // namespace bemcub
