// Step a5 of the hot path: dense BEM collocation matrix,
//     A_ij = k Int_{element j} dS / |c_i - Q|   (unit sigma),  c_i = centroid of element i,
// each entry by the rule its distance ratio DR(i,j) = |c_i - c_j| / L_j asks for (L159), the
// analytic integral below the first limit (self term: D = 0).
//
// Same execution model as the evaluation kernels (kernels_eval.cuh): persistent CTAs, every warp
// pulls items from an atomic queue (12 warps per SM).  One item = (tile of 128 rows) x (split of the
// columns).  A lane owns rows i0 + r * 32 + lane, r < 4 (their centroids sit in registers); the 32 rows
// of one r are a "row group".  Columns are taken 32 at a time: lane l classifies column j0 + l against
// the bounding sphere of the tile's centroids.  Where the whole tile falls into one distance-ratio band
// the column has one rule; where it straddles a limit, the lane classifies the column against the sphere
// of each row group, and the column is streamed once per rule its groups ask for, each copy applied to
// those groups' rows only (or, without allow_upgrade, the column takes the exact per-pair choice with
// masks).  The point records of the batch's columns are streamed through the warp's double-buffered
// shared-memory window by bulk TMA, whole elements per stage, with a small segment table (column, row
// groups, first point, number of points) beside each stage.
//
// The kernel is bound by the issue port, so everything around the 12 FP64
// instructions of an interaction is kept short:
//  * the elements are expanded with k folded into the charges and padded with zero charges to a
//    multiple of kAsmU points, so a column is whole trips of kAsmU points and its sum needs neither a
//    remainder loop nor a final scaling;
//  * results of 8 consecutive columns go through a 128 x 8 shared-memory tile and leave as 64-byte row
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
  const uint32_t* row_perm;   // [nrows] or null: the k-th row of the call, in tile order, is row0 + row_perm[k]
  const int* use_perm;        // device flag (choose_row_order_kernel): take row_perm, or the rows as they come
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
  uint32_t seg[kStages][32];  // col | row-group mask << 5 | npts << 9 | first << 16
  double sub[kAsmR][4];       // bounding spheres of the tile's 32-row groups (centre, radius)
  uint32_t rowidx[kAsmRows];  // rows of the tile, relative to row0 (tiles take the rows in Morton order of their centroids)
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

// The same for NR < 4 of the lane's rows (the rows of the row groups that take this rule; the other
// groups of the column take another one, see the classification below), handed over in a compact copy.
// Fewer rows per lane, more points per trip: 4 - 8 chains as well.  Only tiles of an upgrading policy
// come here, so the per-pair results (allow_upgrade = 0), which promise not to depend on the tile, never do.
template <int NR>
__device__ __forceinline__ void phi_segment_rows(const double4* __restrict__ pts, int npts, const double (&qx)[NR],
                                                 const double (&qy)[NR], const double (&qz)[NR], double (&acc)[NR], double c375) {
  constexpr int U = NR >= 3 ? 2 : 4;  // npts is a multiple of kAsmU = 2: a U = 4 loop may leave one pair
  static_assert(kAsmU == 2, "phi_segment_rows takes pairs of points");
  double part[U][NR];
#pragma unroll
  for (int u = 0; u < U; ++u)
#pragma unroll
    for (int r = 0; r < NR; ++r) part[u][r] = 0.0;
  int i = 0;
#pragma unroll 1
  for (; i + U <= npts; i += U) {
    double4 s[U];
#pragma unroll
    for (int u = 0; u < U; ++u) s[u] = pts[i + u];
#pragma unroll
    for (int u = 0; u < U; ++u)
#pragma unroll
      for (int r = 0; r < NR; ++r) part[u][r] = phi_one(s[u], s[u].w, qx[r], qy[r], qz[r], part[u][r], c375);
  }
  if (U == 4 && i < npts) {
    const double4 s0 = pts[i], s1 = pts[i + 1];
#pragma unroll
    for (int r = 0; r < NR; ++r) {
      part[0][r] = phi_one(s0, s0.w, qx[r], qy[r], qz[r], part[0][r], c375);
      part[1][r] = phi_one(s1, s1.w, qx[r], qy[r], qz[r], part[1][r], c375);
    }
  }
#pragma unroll
  for (int r = 0; r < NR; ++r) {
    if constexpr (U == 4) acc[r] = (part[0][r] + part[1][r]) + (part[2][r] + part[3][r]);
    else acc[r] = part[0][r] + part[1][r];
  }
}
// row `i` of the lane's four (a warp-uniform index)
__device__ __forceinline__ double pick_row(const double (&v)[kAsmR], int i) {
  static_assert(kAsmR == 4, "pick_row: four rows per lane");
  const double lo = (i & 1) ? v[1] : v[0], hi = (i & 1) ? v[3] : v[2];
  return (i & 2) ? hi : lo;
}

// Which order of the rows gives the tighter 32-row groups: the caller's, or the Morton order of the centroids?
// group_radius_kernel: one warp per group and order, radius of the group's bounding sphere (about the centre of
// its FP32 box); choose_row_order_kernel: one warp adds the radii of each order in a fixed sequence and sets the
// flag if Morton order is clearly tighter (a mesh that arrives spatially ordered keeps its order: its groups
// are as compact and its rows lie next to each other in the output).
__global__ void group_radius_kernel(int64_t nrows, const double4* __restrict__ cen, const uint32_t* __restrict__ perm,
                                    int64_t ngroups, float* __restrict__ radius) {
  const int64_t w = (blockIdx.x * (int64_t)blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  if (w >= 2 * ngroups) return;
  const int which = w >= ngroups;
  const int64_t g = which ? w - ngroups : w;
  const int64_t k = min(g * 32 + lane, nrows - 1);
  const double4 c = cen[which ? (int64_t)perm[k] : k];
  const float fx = (float)c.x, fy = (float)c.y, fz = (float)c.z;
  const double sx = 0.5 * ((double)warp_min_f32(fx) + (double)warp_max_f32(fx));
  const double sy = 0.5 * ((double)warp_min_f32(fy) + (double)warp_max_f32(fy));
  const double sz = 0.5 * ((double)warp_min_f32(fz) + (double)warp_max_f32(fz));
  const double d2 = (c.x - sx) * (c.x - sx) + (c.y - sy) * (c.y - sy) + (c.z - sz) * (c.z - sz);
  const float r = sqrtf(warp_max_f32((float)d2));
  if (lane == 0) radius[w] = r;
}
__global__ void choose_row_order_kernel(int64_t ngroups, const float* __restrict__ radius, int* __restrict__ use_perm) {
  const int lane = threadIdx.x;
  double s[2] = {0.0, 0.0};
  for (int which = 0; which < 2; ++which) {
    for (int64_t g = lane; g < ngroups; g += 32) s[which] += (double)radius[which * ngroups + g];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s[which] += __shfl_xor_sync(kFullMask, s[which], o);
  }
  if (lane == 0) *use_perm = s[1] < 0.8 * s[0];
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
    // The queue is run through twice.  The first pass takes the expensive column batches of an item
    // (near the tile: 19 points and more per column, analytic entries, several rules per column), the
    // second pass the cheap rest, so the launch ends on items of equal, small cost: its tail (the warps
    // that find the queue empty while others still work) is half a cheap item instead of half an expensive one.
    int64_t item = next_item(p.queue, lane);
    if (item >= 2 * p.nitems) break;
    const bool second_pass = item >= p.nitems;
    if (second_pass) item -= p.nitems;
    const int64_t split = item / p.nrowtiles, rt = item - split * p.nrowtiles;
    const int64_t r0 = rt * kAsmRows;  // first row of the tile in tile order
    const bool use_perm = p.row_perm && *p.use_perm;
    const int nrow_here = (int)min((int64_t)kAsmRows, p.nrows - r0);

    // rows: field points = centroids (clamped duplicates compute harmlessly and are never stored)
    double px[kAsmR], py[kAsmR], pz[kAsmR];
    bool ok[kAsmR];
#pragma unroll
    for (int r = 0; r < kAsmR; ++r) {
      ok[r] = r * 32 + lane < nrow_here;
      const int64_t k = r0 + min(r * 32 + lane, nrow_here - 1);
      const uint32_t row = use_perm ? p.row_perm[k] : (uint32_t)k;
      sm.rowidx[r * 32 + lane] = row;
      const double4 ci = p.cenL[p.row0 + row];
      px[r] = ci.x; py[r] = ci.y; pz[r] = ci.z;
    }
    // Bounding spheres of every 32-row group (rows r * 32 + lane: consecutive elements, a compact patch of
    // a spatially ordered mesh; kept in shared memory) and of the whole tile.  The boxes are taken in FP32
    // (one REDUX per bound): any centre will do as long as the radius about it is not under-estimated, so
    // the radius is the FP64 distance of the farthest centroid, rounded up on its way through FP32.
    float lox = CUDART_INF_F, hix = -CUDART_INF_F, loy = CUDART_INF_F, hiy = -CUDART_INF_F, loz = CUDART_INF_F, hiz = -CUDART_INF_F;
    __syncwarp();
#pragma unroll
    for (int r = 0; r < kAsmR; ++r) {
      const float fx = (float)px[r], fy = (float)py[r], fz = (float)pz[r];
      const float ax = warp_min_f32(fx), bx = warp_max_f32(fx), ay = warp_min_f32(fy), by = warp_max_f32(fy);
      const float az = warp_min_f32(fz), bz = warp_max_f32(fz);
      const double sx = 0.5 * ((double)ax + (double)bx), sy = 0.5 * ((double)ay + (double)by), sz = 0.5 * ((double)az + (double)bz);
      const double s2 = (px[r] - sx) * (px[r] - sx) + (py[r] - sy) * (py[r] - sy) + (pz[r] - sz) * (pz[r] - sz);
      const float srho = __fsqrt_ru(warp_max_f32(__double2float_ru(s2)));
      if (lane == 0) {
        sm.sub[r][0] = sx; sm.sub[r][1] = sy; sm.sub[r][2] = sz; sm.sub[r][3] = (double)srho;
      }
      lox = fminf(lox, ax); hix = fmaxf(hix, bx);
      loy = fminf(loy, ay); hiy = fmaxf(hiy, by);
      loz = fminf(loz, az); hiz = fmaxf(hiz, bz);
    }
    __syncwarp();
    const double cx = 0.5 * ((double)lox + (double)hix), cy = 0.5 * ((double)loy + (double)hiy), cz = 0.5 * ((double)loz + (double)hiz);
    double d2 = 0.0;
#pragma unroll
    for (int r = 0; r < kAsmR; ++r)
      d2 = fmax(d2, (px[r] - cx) * (px[r] - cx) + (py[r] - cy) * (py[r] - cy) + (pz[r] - cz) * (pz[r] - cz));
    const double rho = (double)__fsqrt_ru(warp_max_f32(__double2float_ru(d2)));
    const double mag = fmax(fmax(fabs(cx), fabs(cy)), fabs(cz)) + rho;
    // valid rows of each group, one byte per group (for the interaction tally)
    uint32_t vrows = 0;
#pragma unroll
    for (int r = 0; r < kAsmR; ++r) vrows |= (uint32_t)max(0, min(32, nrow_here - 32 * r)) << (8 * r);

    // analytic pair queue of this item: [aq_head, aq_tail) in the ring sm.aq
    int aq_head = 0, aq_tail = 0;
    // Evaluates `take` (<= 32) queued pairs, one per lane: entry = row << 25 | column.
    auto drain = [&](int take) {
      __syncwarp();
      if (lane < take) {
        const uint32_t ent = sm.aq[(aq_head + lane) & (kAqCap - 1)];
        const int row = (int)(ent >> 25);
        const int64_t col = (int64_t)(ent & 0x1ffffffu);
        const int64_t grow = sm.rowidx[row];
        const double4 ci = ldg4(p.cenL + p.row0 + grow);
        Vec3 V[4];
        const int nv = load_polygon(p.type, p.verts, col, V);
        double ip;
        Vec3 ie;
        analytic_integrals<false>(V, nv, Vec3{ci.x, ci.y, ci.z}, ip, ie);
        p.out[grow * p.ld + col] = p.k * ip;
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
      // lm: which row groups take which cubature level, 4 bits per level (bit 4 L + r: group r, level L).
      // A column the whole tile sees in one band has one level with all four groups; where the tile
      // straddles a band limit (and the policy allows upgrades) every 32-row group is classified by its own
      // sphere, so the more accurate rule is paid by the groups that need it only.
      uint32_t lm = 0;
      int cnt = 0, lvl = -1;  // cnt: the column's points in the stream (all its levels), zero-charge padding included
      int real = 0;           // point-charge interactions of the column with the valid rows, without the padding
      int nseg = 0;           // levels of the column = its segments in the stream
      bool has_ana = false, is_mixed = false;
      const double4* src = nullptr;
      int t = 0;
      if (lane < ncol) {
        const double4 c = p.cenL[e];
        t = p.type[e];
        const double cmag = fmax(fmax(fabs(c.x), fabs(c.y)), fabs(c.z));
        const double dx = cx - c.x, dy = cy - c.y, dz = cz - c.z;
        const double Dc = sqrt(dx * dx + dy * dy + dz * dz);
        const double slack = 1e-9 * (Dc + rho) + 1e-12 * (mag + cmag);
        const double Dhi = Dc + rho + slack, Dlo = fmax(Dc - rho - slack, 0.0);
        const int lfar = p.pol.map[want_level(Dhi * Dhi, c.w, p.pol.dr[t])];
        const int lnear = p.pol.map[want_level(Dlo * Dlo, c.w, p.pol.dr[t])];
        if (lnear == lfar) {
          if (lnear == 5) has_ana = true;  // every row below the analytic limit: nothing streamed
          else lm = 0xfu << (4 * lnear);
        } else if (!p.pol.allow_upgrade) {
          is_mixed = true;  // exact per-pair choice
        } else {
          // The analytic formula is never an "upgrade" (see eval_adaptive_kernel).  A group that
          // straddles the analytic limit is streamed with the most accurate cubature rule and its
          // rows below the limit are overwritten analytically afterwards; a group entirely below the
          // limit is not streamed at all.
#pragma unroll 1
          for (int r = 0; r < kAsmR; ++r) {
            const double sx = sm.sub[r][0] - c.x, sy = sm.sub[r][1] - c.y, sz = sm.sub[r][2] - c.z, srho = sm.sub[r][3];
            const double Ds = sqrt(sx * sx + sy * sy + sz * sz);
            const double sl = 1e-9 * (Ds + srho) + 1e-12 * (mag + cmag);
            const double Shi = Ds + srho + sl, Slo = fmax(Ds - srho - sl, 0.0);
            const int gfar = p.pol.map[want_level(Shi * Shi, c.w, p.pol.dr[t])];
            const int gnear = p.pol.map[want_level(Slo * Slo, c.w, p.pol.dr[t])];
            if (gnear == 5) {
              has_ana = true;
              if (gfar != 5) {
                if (p.pol.map[4] == 5) is_mixed = true;  // no cubature level to fall back on
                else lm |= 1u << (4 * p.pol.map[4] + r);
              }
            } else {
              lm |= 1u << (4 * gnear + r);
            }
          }
          if (is_mixed) {
            lm = 0;
            has_ana = false;
          }
        }
#pragma unroll
        for (int L = 0; L < 5; ++L) {
          const uint32_t g = (lm >> (4 * L)) & 15u;
          if (g) {
            const int N = rule_npts(t, L);
            cnt += (N + kAsmU - 1) / kAsmU * kAsmU;
            real += N * (int)__dp4a(vrows, ((g & 1u) | ((g & 2u) << 7) | ((g & 4u) << 14) | ((g & 8u) << 21)), 0u);
            lvl = nseg ? -2 : L;  // -2: several levels, its copies are never merged with a neighbour's
            src = p.lvl_pts[L] + e * p.stride[L];
            ++nseg;
          }
        }
      }
      const bool costly = __any_sync(kFullMask, lvl >= 3 || lvl == -2 || has_ana || is_mixed);
      if (costly == second_pass) continue;
      // point-charge interactions of the batch's streamed columns (padding and clamped rows not counted)
      const int real_pts = warp_sum(real);
      if (lane == 0) sm.n_inter += (unsigned long long)real_pts;
      int total, ktotal;
      const int pre = warp_excl_scan(cnt, lane, &total);
      const int kpre = warp_excl_scan(nseg, lane, &ktotal);
      int cursor = 0;

      // Fills `stage` with the next whole elements of the batch; returns how many (0 = batch done).
      auto fill = [&](int stage) -> int {
        for (;;) {
          if (cursor >= 32) return 0;
          const int kbase = __shfl_sync(kFullMask, kpre, cursor);
          const StagePlan sp = plan_stage(cursor, lane, cnt, pre, total, lvl, p.stride);
          cursor = sp.next;
          if (sp.nstage == 0) continue;
          const int kend = __shfl_sync(kFullMask, kpre, sp.next & 31);
          const uint32_t dst = win0 + (uint32_t)((stage * kBuf + (pre - sp.base)) * sizeof(double4));
          if (lane == 0) mbar_arrive_expect_tx(bar0 + 8 * stage, (uint32_t)(sp.nstage * sizeof(double4)));
          if (sp.inc && lvl >= 0)
            sm.seg[stage][kpre - kbase] = (uint32_t)lane | (((lm >> (4 * lvl)) & 15u) << 5) | ((uint32_t)cnt << 9) | ((uint32_t)(pre - sp.base) << 16);
          __syncwarp();
          if (sp.inc) {
            if (lvl >= 0) {  // one level: consecutive columns share a copy
              if (sp.head) tma_load_1d(dst, src, (uint32_t)((sp.run_end - pre) * sizeof(double4)), bar0 + 8 * stage);
            } else {  // one segment and one copy per level, the most accurate first
              int k = kpre - kbase, off = 0;
              for (int L = 4; L >= 0; --L) {
                const uint32_t g = (lm >> (4 * L)) & 15u;
                if (!g) continue;
                const int np = (rule_npts(t, L) + kAsmU - 1) / kAsmU * kAsmU;
                sm.seg[stage][k++] = (uint32_t)lane | (g << 5) | ((uint32_t)np << 9) | ((uint32_t)(pre - sp.base + off) << 16);
                tma_load_1d(dst + (uint32_t)(off * sizeof(double4)), p.lvl_pts[L] + e * p.stride[L], (uint32_t)(np * sizeof(double4)),
                            bar0 + 8 * stage);
                off += np;
              }
            }
          }
          __syncwarp();  // the segment table is complete before any lane reads it
          return (sp.next < 32 ? kend : ktotal) - kbase;
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
                double2* o = reinterpret_cast<double2*>(p.out + (int64_t)sm.rowidx[row] * p.ld + jg);
                const double2 a = make_double2(t[0], t[kAsmRows]), b = make_double2(t[2 * kAsmRows], t[3 * kAsmRows]);
                const double2 c = make_double2(t[4 * kAsmRows], t[5 * kAsmRows]), d = make_double2(t[6 * kAsmRows], t[7 * kAsmRows]);
                o[0] = a; o[1] = b; o[2] = c; o[3] = d;
              }
            }
          } else {
            const int c = lane & (kGroupCols - 1);
            if ((gmask >> c) & 1u) {
              const double* t = &sm.tile[c * kAsmRows + (lane >> 3)];
              for (int row = lane >> 3; row < nrow_here; row += 4, t += 4) p.out[(int64_t)sm.rowidx[row] * p.ld + jg + c] = *t;
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
          const double4* pts = &sm.win[stage][d >> 16];
          const int npts = (int)((d >> 9) & 127u);
          __builtin_assume(npts >= kAsmU);  // a segment is never empty
          const uint32_t g = (d >> 5) & 15u;
          double* trow = &sm.tile[(col & (kGroupCols - 1)) * kAsmRows + lane];
          if (g == 15u) {
            double acc[kAsmR];
            phi_segment(pts, npts, px, py, pz, acc, c375);
#pragma unroll
            for (int r = 0; r < kAsmR; ++r) trow[r * 32] = acc[r];
          } else if (__popc(g) == 3) {  // all rows but one
            const int skip = __ffs(~g) - 1;
            double qx[3], qy[3], qz[3], acc[3];
#pragma unroll
            for (int i = 0; i < 3; ++i) {
              qx[i] = i < skip ? px[i] : px[i + 1];
              qy[i] = i < skip ? py[i] : py[i + 1];
              qz[i] = i < skip ? pz[i] : pz[i + 1];
            }
            phi_segment_rows<3>(pts, npts, qx, qy, qz, acc, c375);
#pragma unroll
            for (int i = 0; i < 3; ++i) trow[(i < skip ? i : i + 1) * 32] = acc[i];
          } else if (__popc(g) == 2) {
            const int i0 = __ffs(g) - 1, i1 = 31 - __clz(g);
            const double qx[2] = {pick_row(px, i0), pick_row(px, i1)}, qy[2] = {pick_row(py, i0), pick_row(py, i1)};
            const double qz[2] = {pick_row(pz, i0), pick_row(pz, i1)};
            double acc[2];
            phi_segment_rows<2>(pts, npts, qx, qy, qz, acc, c375);
            trow[i0 * 32] = acc[0];
            trow[i1 * 32] = acc[1];
          } else {
            const int i0 = __ffs(g) - 1;
            const double qx[1] = {pick_row(px, i0)}, qy[1] = {pick_row(py, i0)}, qz[1] = {pick_row(pz, i0)};
            double acc[1];
            phi_segment_rows<1>(pts, npts, qx, qy, qz, acc, c375);
            trow[i0 * 32] = acc[0];
          }
          gmask |= 1u << (col & (kGroupCols - 1));
        }
        __syncwarp();
      };

      // the columns that need the exact per-pair choice (none under an upgrading policy), stored directly
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
          if (ok[r]) p.out[(int64_t)sm.rowidx[r * 32 + lane] * p.ld + j] = val[r];
      }
      // ---- streamed columns: fill the other stage, then consume this one (one call site each: the
      // kernel has to fit the instruction cache)
      for (int stage = 1, cur = 0;;) {
        const int nxt = fill(stage ^ 1);
        if (cur > 0) consume_stage(stage, cur);
        if (nxt == 0) break;
        stage ^= 1;
        cur = nxt;
      }
      flush_group();
      // ---- entries below the analytic limit: every row of a column the whole tile (or a row group) sees
      // that near, and - by the exact per-pair test - the rows of the straddling groups streamed above
      // (their cubature values are overwritten: flush_group has synchronised the warp).  Queued, then
      // evaluated one pair per lane.
      unsigned qmask = __ballot_sync(kFullMask, has_ana);
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
