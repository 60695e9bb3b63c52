// Step a5 of the hot path: dense BEM collocation matrix,
//     A_ij = k Int_{element j} dS / |c_i - Q|   (unit sigma),  c_i = centroid of element i,
// each entry by the rule its distance ratio DR(i,j) = |c_i - c_j| / L_j asks for (L159), the
// analytic integral below the first limit (self term: D = 0).
//
// Same execution model as the evaluation kernels (kernels_eval.cuh): persistent CTAs, every warp
// pulls items from an atomic queue (16 warps per SM here).  One item = (tile of 64 rows) x (split of
// the columns).  A lane owns rows i0 + lane and i0 + 32 + lane (their centroids sit in registers).
// Columns are taken 32 at a time: lane l classifies column j0+l against the bounding sphere of the
// row centroids, so the rule of a column is warp-uniform unless the tile straddles a band limit
// (then: the more accurate rule, or the exact per-pair choice with masks).  The point records of the
// batch's columns are streamed through the warp's double-buffered shared-memory window by bulk TMA,
// whole elements per stage, with a small segment table (column, first point, number of points)
// beside each stage.
//
// The kernel is bound by the issue port, so everything around the 12 FP64
// instructions of an interaction is kept short:
//  * the elements are expanded with k folded into the charges and padded with zero charges to a
//    multiple of kAsmU points, so a column is whole trips of kAsmU points and its sum needs neither a
//    remainder loop nor a final scaling;
//  * results of 8 consecutive columns go through a 64 x 8 shared-memory tile and leave as 64-byte row
//    segments, each lane storing its own rows with four 16-byte stores;
//  * entries below the analytic limit are not evaluated where they are met (a warp-wide call for a
//    handful of rows): their (row, column) pairs are queued in shared memory and evaluated 32 at a
//    time, one pair per lane.
#pragma once
#include "kernels_eval.cuh"

namespace bemcub {

struct AssembleParams {
  const double4* lvl_pts[5];  // unit-sigma points per level, charges times k, padded (see above)
  int stride[5];
  const double4* cenL;
  const uint8_t* type;
  const double* verts;
  int64_t n;
  PolicyDev pol;
  int64_t row0, nrows;
  double* out;
  int64_t ld;
  double k;
  int64_t cols_per_split;     // multiple of 32
  int64_t nrowtiles, nitems;  // item = split * nrowtiles + rowtile
  unsigned long long* queue;
  unsigned long long* counters;
};

// Measured on config 3 (round 2): 4 rows per lane x 2 points per trip at 12 warps/SM 5.65 ms, 2 x 4 at 16
// warps 5.80 ms, 2 x 4 at 12 warps 5.76 ms, 4 x 1 at 12 warps 6.20 ms.
constexpr int kAsmWarps = 12;
constexpr int kAsmThreads = kAsmWarps * 32;
constexpr int kAsmR = 4;               // rows per lane
constexpr int kAsmU = 2;               // points per trip; the expanded elements are padded to a multiple of it
constexpr int kAsmRows = 32 * kAsmR;   // rows per tile
constexpr int kGroupCols = 8;          // columns per output group: 64-byte row segments = two full sectors
constexpr int kAqCap = kAsmR <= 2 ? 128 : 256;  // analytic pair queue (ring, >= 32 + 32 kAsmR), entries = row << 25 | column
constexpr int64_t kAsmMaxN = (int64_t)1 << 25;  // ... hence this many elements at most (a 2^26-square matrix is out of reach anyway)

// per-warp shared memory: window | output tile | segment tables | analytic queue | mbarriers | tallies
struct AsmWarpSmem {
  double4 win[kStages][kBuf];
  double tile[kGroupCols * kAsmRows];  // [column of the group][row]: conflict-free both ways
  uint32_t seg[kStages][32];  // col | npts << 8 | first << 16
  uint32_t aq[kAqCap];
  uint64_t bar[kStages];
  unsigned long long n_inter, n_ana;
};
constexpr size_t assemble_smem_bytes() { return (size_t)kAsmWarps * sizeof(AsmWarpSmem); }

// Potential-only term of Eq. 4.1: 12 FP64-pipe instructions (3 DADD + 3 DMUL + 6 DFMA).
__device__ __forceinline__ double phi_one(const double4 s, double q, double px, double py, double pz, double acc, double c375) {
  const double dx = __dsub_rn(px, s.x), dy = __dsub_rn(py, s.y), dz = __dsub_rn(pz, s.z);
  const double r2 = __fma_rn(dx, dx, __fma_rn(dy, dy, __dmul_rn(dz, dz)));
  return __fma_rn(q, rsqrt_f64(r2, dz, c375), acc);
}

// One element's points (already in shared memory; npts a multiple of kAsmU thanks to the zero-charge
// padding) against the lane's kAsmR rows, kAsmU points per trip with their own partial sums:
// kAsmU * kAsmR = 8 independent chains per lane.
__device__ __forceinline__ void phi_segment(const double4* __restrict__ pts, int npts, const double (&px)[kAsmR],
                                            const double (&py)[kAsmR], const double (&pz)[kAsmR], double (&acc)[kAsmR],
                                            double c375) {
  constexpr int U = kAsmU;
  double part[U][kAsmR];
#pragma unroll
  for (int u = 0; u < U; ++u)
#pragma unroll
    for (int r = 0; r < kAsmR; ++r) part[u][r] = 0.0;
#pragma unroll 1
  for (int i = 0; i < npts; i += U) {
    double4 s[U];
#pragma unroll
    for (int u = 0; u < U; ++u) s[u] = pts[i + u];
#pragma unroll
    for (int u = 0; u < U; ++u)
#pragma unroll
      for (int r = 0; r < kAsmR; ++r) part[u][r] = phi_one(s[u], s[u].w, px[r], py[r], pz[r], part[u][r], c375);
  }
#pragma unroll
  for (int r = 0; r < kAsmR; ++r) {
    if constexpr (U == 4) acc[r] = (part[0][r] + part[1][r]) + (part[2][r] + part[3][r]);
    else if constexpr (U == 2) acc[r] = part[0][r] + part[1][r];
    else acc[r] = part[0][r];
  }
}

__global__ void __launch_bounds__(kAsmThreads, 1) assemble_kernel(const __grid_constant__ AssembleParams p) {
  static_assert(kAsmU == 4 || kAsmU == 2 || kAsmU == 1, "phi_segment's sum tree");
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  AsmWarpSmem& sm = reinterpret_cast<AsmWarpSmem*>(smem_raw)[warp];
  const uint32_t bar0 = smem_u32(&sm.bar[0]), win0 = smem_u32(&sm.win[0][0]);
  if (lane == 0) {
    mbar_init(bar0, 1);
    mbar_init(bar0 + 8, 1);
    mbar_fence_init();
    sm.n_inter = 0;
    sm.n_ana = 0;
  }
  __syncwarp();
  uint32_t phases = 0;
  const unsigned lt_mask = (1u << lane) - 1u;
  const double c375 = c_three_eighths;
  // 16-byte stores of whole 8-column groups need even ld and an aligned base
  const bool vec_ok = ((p.ld & 1) == 0) && ((reinterpret_cast<uintptr_t>(p.out) & 15u) == 0);
  KernelClock clk;
  clk.begin();

  for (;;) {
    const int64_t item = next_item(p.queue, lane);
    if (item >= p.nitems) break;
    const int64_t split = item / p.nrowtiles, rt = item - split * p.nrowtiles;
    const int64_t r0 = rt * kAsmRows;  // first row of the tile, relative to row0
    const int nrow_here = (int)min((int64_t)kAsmRows, p.nrows - r0);

    // rows: field points = centroids (clamped duplicates compute harmlessly and are never stored)
    double px[kAsmR], py[kAsmR], pz[kAsmR];
    bool ok[kAsmR];
#pragma unroll
    for (int r = 0; r < kAsmR; ++r) {
      ok[r] = r * 32 + lane < nrow_here;
      const double4 ci = p.cenL[p.row0 + r0 + min(r * 32 + lane, nrow_here - 1)];
      px[r] = ci.x; py[r] = ci.y; pz[r] = ci.z;
    }
    double lox = px[0], hix = px[0], loy = py[0], hiy = py[0], loz = pz[0], hiz = pz[0];
#pragma unroll
    for (int r = 1; r < kAsmR; ++r) {
      lox = fmin(lox, px[r]); hix = fmax(hix, px[r]);
      loy = fmin(loy, py[r]); hiy = fmax(hiy, py[r]);
      loz = fmin(loz, pz[r]); hiz = fmax(hiz, pz[r]);
    }
    lox = warp_min(lox); hix = warp_max(hix);
    loy = warp_min(loy); hiy = warp_max(hiy);
    loz = warp_min(loz); hiz = warp_max(hiz);
    const double cx = 0.5 * (lox + hix), cy = 0.5 * (loy + hiy), cz = 0.5 * (loz + hiz);
    double d2 = 0.0;
#pragma unroll
    for (int r = 0; r < kAsmR; ++r)
      d2 = fmax(d2, (px[r] - cx) * (px[r] - cx) + (py[r] - cy) * (py[r] - cy) + (pz[r] - cz) * (pz[r] - cz));
    const double rho = sqrt(warp_max(d2));
    const double mag = fmax(fmax(fabs(cx), fabs(cy)), fabs(cz)) + rho;

    // analytic pair queue of this item: [aq_head, aq_tail) in the ring sm.aq
    int aq_head = 0, aq_tail = 0;
    // Evaluates `take` (<= 32) queued pairs, one per lane: entry = row << 25 | column.
    auto drain = [&](int take) {
      __syncwarp();
      if (lane < take) {
        const uint32_t ent = sm.aq[(aq_head + lane) & (kAqCap - 1)];
        const int row = (int)(ent >> 25);
        const int64_t col = (int64_t)(ent & 0x1ffffffu);
        const double4 ci = ldg4(p.cenL + p.row0 + r0 + row);
        Vec3 V[4];
        const int nv = load_polygon(p.type, p.verts, col, V);
        double ip;
        Vec3 ie;
        analytic_integrals<false>(V, nv, Vec3{ci.x, ci.y, ci.z}, ip, ie);
        p.out[(r0 + row) * p.ld + col] = p.k * ip;
      }
      aq_head += take;
      __syncwarp();
    };

    const int64_t col_begin = split * p.cols_per_split;
    const int64_t col_end = min(p.n, col_begin + p.cols_per_split);
    for (int64_t j0 = col_begin; j0 < col_end; j0 += 32) {
      const int ncol = (int)min((int64_t)32, col_end - j0);
      // ---- classify column j0 + lane against the row tile's bounding sphere
      const int64_t e = j0 + lane;
      int cnt = 0, lvl = -1;  // cnt: the column's points in the stream, zero-charge padding included
      int real = 0;           // ... and without it
      bool is_ana = false, is_mixed = false, is_fix = false;
      const double4* src = nullptr;
      if (lane < ncol) {
        const double4 c = p.cenL[e];
        const int t = p.type[e];
        const double dx = cx - c.x, dy = cy - c.y, dz = cz - c.z;
        const double Dc = sqrt(dx * dx + dy * dy + dz * dz);
        const double slack = 1e-9 * (Dc + rho) + 1e-12 * (mag + fmax(fmax(fabs(c.x), fabs(c.y)), fabs(c.z)));
        const double Dhi = Dc + rho + slack, Dlo = fmax(Dc - rho - slack, 0.0);
        const int lfar = p.pol.map[want_level(Dhi * Dhi, c.w, p.pol.dr[t])];
        const int lnear = p.pol.map[want_level(Dlo * Dlo, c.w, p.pol.dr[t])];
        // the analytic formula is never an "upgrade" (see eval_adaptive_kernel): a tile straddling
        // the analytic limit keeps the exact per-pair choice
        if (lnear != lfar && lnear == 5 && p.pol.allow_upgrade && p.pol.map[4] != 5) {
          // tile straddles the analytic limit: the column is streamed with the most accurate
          // cubature rule, and the rows below the limit are overwritten analytically afterwards
          is_fix = true;
          lvl = p.pol.map[4];
        } else if (lnear != lfar && (!p.pol.allow_upgrade || lnear == 5)) {
          is_mixed = true;
        } else {
          lvl = lnear;
          is_ana = lvl == 5;
        }
        if (lvl >= 0 && lvl < 5) {
          real = rule_npts(t, lvl);
          cnt = (real + kAsmU - 1) / kAsmU * kAsmU;
          src = p.lvl_pts[lvl] + e * p.stride[lvl];
        }
      }
      // point-charge interactions of the batch's streamed columns (padding not counted)
      const int real_pts = warp_sum(real);
      if (lane == 0) sm.n_inter += (unsigned long long)real_pts * nrow_here;
      int total;
      const int pre = warp_excl_scan(cnt, lane, &total);
      int cursor = 0;

      // Fills `stage` with the next whole elements of the batch; returns how many (0 = batch done).
      auto fill = [&](int stage) -> int {
        for (;;) {
          if (cursor >= 32) return 0;
          const StagePlan sp = plan_stage(cursor, lane, cnt, pre, total, lvl, p.stride);
          cursor = sp.next;
          if (sp.nstage == 0) continue;
          if (sp.inc) sm.seg[stage][__popc(sp.incmask & lt_mask)] = (uint32_t)lane | ((uint32_t)cnt << 8) | ((uint32_t)(pre - sp.base) << 16);
          if (lane == 0) mbar_arrive_expect_tx(bar0 + 8 * stage, (uint32_t)(sp.nstage * sizeof(double4)));
          __syncwarp();
          if (sp.head)
            tma_load_1d(win0 + (uint32_t)((stage * kBuf + (pre - sp.base)) * sizeof(double4)), src,
                        (uint32_t)((sp.run_end - pre) * sizeof(double4)), bar0 + 8 * stage);
          return __popc(sp.incmask);
        }
      };
      // output group (8 consecutive columns) being collected in sm.tile, and which of its columns
      int cur_group = -1;
      unsigned gmask = 0;
      auto flush_group = [&]() {
        __syncwarp();
        if (cur_group >= 0) {
          const int64_t jg = j0 + cur_group * kGroupCols;
          if (gmask == 0xffu && vec_ok) {
            // all 8 columns present: every lane stores the 64 bytes of each of its rows
#pragma unroll
            for (int r = 0; r < kAsmR; ++r) {
              const int row = r * 32 + lane;
              if (row < nrow_here) {
                const double* t = &sm.tile[row];
                double2* o = reinterpret_cast<double2*>(p.out + (r0 + row) * p.ld + jg);
                const double2 a = make_double2(t[0], t[kAsmRows]), b = make_double2(t[2 * kAsmRows], t[3 * kAsmRows]);
                const double2 c = make_double2(t[4 * kAsmRows], t[5 * kAsmRows]), d = make_double2(t[6 * kAsmRows], t[7 * kAsmRows]);
                o[0] = a; o[1] = b; o[2] = c; o[3] = d;
              }
            }
          } else {
            const int c = lane & (kGroupCols - 1);
            if ((gmask >> c) & 1u) {
              double* o = p.out + (r0 + (lane >> 3)) * p.ld + jg + c;
              const double* t = &sm.tile[c * kAsmRows + (lane >> 3)];
              for (int row = lane >> 3; row < nrow_here; row += 4, o += 4 * p.ld, t += 4) *o = *t;
            }
          }
        }
        __syncwarp();
      };
      auto consume_stage = [&](int stage, int nseg) {
        mbar_wait(bar0 + 8 * stage, (phases >> stage) & 1u);
        phases ^= 1u << stage;
        for (int k = 0; k < nseg; ++k) {
          const uint32_t d = sm.seg[stage][k];
          const int col = (int)(d & 31u);
          if ((col >> 3) != cur_group) {
            flush_group();
            cur_group = col >> 3;
            gmask = 0;
          }
          double acc[kAsmR];
          phi_segment(&sm.win[stage][d >> 16], (int)((d >> 8) & 255u), px, py, pz, acc, c375);
#pragma unroll
          for (int r = 0; r < kAsmR; ++r) sm.tile[(col & (kGroupCols - 1)) * kAsmRows + r * 32 + lane] = acc[r];
          gmask |= 1u << (col & (kGroupCols - 1));
        }
        __syncwarp();
      };

      int na = fill(0);
      int nb = na ? fill(1) : 0;
      // while the first copies fly: the rare columns that need the exact per-pair choice, stored directly
      unsigned xmask = __ballot_sync(kFullMask, is_mixed);
      while (xmask) {
        const int l = __ffs(xmask) - 1;
        xmask &= xmask - 1;
        const int64_t j = j0 + l;
        const double4 c = ldg4(p.cenL + j);
        const int t = __ldg(p.type + j);
        int lev[kAsmR];
        double val[kAsmR];
#pragma unroll
        for (int r = 0; r < kAsmR; ++r) {
          const double dx = __dsub_rn(px[r], c.x), dy = __dsub_rn(py[r], c.y), dz = __dsub_rn(pz[r], c.z);
          const double D2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
          lev[r] = p.pol.map[want_level(D2, c.w, p.pol.dr[t])];
          val[r] = 0.0;
        }
        for (int lv = 0; lv <= 5; ++lv) {
          bool take[kAsmR];
          bool any = false;
          int mine = 0;
#pragma unroll
          for (int r = 0; r < kAsmR; ++r) {
            take[r] = lev[r] == lv;
            any |= take[r];
            mine += (take[r] && ok[r]) ? 1 : 0;
          }
          if (!__any_sync(kFullMask, any)) continue;
          const int all = warp_sum(mine);
          if (lv == 5) {
            Vec3 V[4];
            const int nv = load_polygon(p.type, p.verts, j, V);
#pragma unroll
            for (int r = 0; r < kAsmR; ++r) {
              if (!take[r]) continue;
              double ip;
              Vec3 ie;
              analytic_integrals<false>(V, nv, Vec3{px[r], py[r], pz[r]}, ip, ie);
              val[r] = p.k * ip;
            }
            if (lane == 0) sm.n_ana += (unsigned long long)all;
          } else {
            // the same arithmetic, in the same order, as the streamed columns (phi_segment on the
            // padded record list, read from global memory here): an entry does not depend on the
            // tile it was computed in
            const int N = rule_npts(t, lv);
            double acc[kAsmR];
            phi_segment(p.lvl_pts[lv] + j * p.stride[lv], (N + kAsmU - 1) / kAsmU * kAsmU, px, py, pz, acc, c375);
#pragma unroll
            for (int r = 0; r < kAsmR; ++r)
              if (take[r]) val[r] = acc[r];
            if (lane == 0) sm.n_inter += (unsigned long long)all * N;
          }
        }
#pragma unroll
        for (int r = 0; r < kAsmR; ++r)
          if (ok[r]) p.out[(r0 + r * 32 + lane) * p.ld + j] = val[r];
      }
      // ---- streamed columns
      for (;;) {
        if (!na) break;
        consume_stage(0, na);
        na = fill(0);
        if (!nb) break;
        consume_stage(1, nb);
        nb = fill(1);
      }
      flush_group();
      // ---- entries below the analytic limit: every row of a column the whole tile sees that near,
      // and - by the exact per-pair test - the rows of the straddling columns streamed above (their
      // cubature values are overwritten: flush_group has synchronised the warp).  Queued, then
      // evaluated one pair per lane.
      unsigned qmask = __ballot_sync(kFullMask, is_ana || is_fix);
      while (qmask) {
        const int l = __ffs(qmask) - 1;
        qmask &= qmask - 1;
        const int64_t j = j0 + l;
        const double4 c = ldg4(p.cenL + j);
        const int t = __ldg(p.type + j);
#pragma unroll
        for (int r = 0; r < kAsmR; ++r) {
          const double dx = __dsub_rn(px[r], c.x), dy = __dsub_rn(py[r], c.y), dz = __dsub_rn(pz[r], c.z);
          const double D2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
          const bool take = ok[r] && p.pol.map[want_level(D2, c.w, p.pol.dr[t])] == 5;
          const unsigned bal = __ballot_sync(kFullMask, take);
          if (take) sm.aq[(aq_tail + __popc(bal & lt_mask)) & (kAqCap - 1)] = ((uint32_t)(r * 32 + lane) << 25) | (uint32_t)j;
          aq_tail += __popc(bal);
        }
        while (aq_tail - aq_head >= 32) drain(32);
      }
    }
    if (lane == 0) sm.n_ana += (unsigned long long)aq_tail;
    if (aq_tail > aq_head) drain(aq_tail - aq_head);
  }

  __syncwarp();
  if (p.counters && lane == 0) {
    if (sm.n_inter) atomicAdd(p.counters, sm.n_inter);
    if (sm.n_ana) atomicAdd(p.counters + 1, sm.n_ana);
  }
  clk.end(p.counters);
}

}  // namespace bemcub
