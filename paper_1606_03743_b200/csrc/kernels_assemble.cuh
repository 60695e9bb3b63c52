// Step a5 of the hot path: dense BEM collocation matrix,
//     A_ij = k Int_{element j} dS / |c_i - Q|   (unit sigma),  c_i = centroid of element i,
// each entry by the rule its distance ratio DR(i,j) = |c_i - c_j| / L_j asks for (L159), the
// analytic integral below the first limit (self term: D = 0).
//
// One warp fills a 32 x 32 tile: lane l owns ROW i0+l (its field point c_i sits in registers) and,
// for the classification, COLUMN j0+l.  Columns are then walked warp-uniformly: the rule of column
// j against the bounding sphere of the 32 row centroids is the same for all lanes unless the tile
// straddles a band limit (then: more accurate rule, or exact per-pair choice with masks).  The
// 32 x 32 results go through a padded shared-memory tile and leave as 32 row segments of 256
// contiguous bytes (coalesced row-major FP64 stores).
#pragma once
#include "kernels_eval.cuh"

namespace bemcub {

struct AssembleParams {
  const double4* lvl_pts[5];  // unit-sigma points per level
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
  unsigned long long* counters;
};

constexpr int kAsmWarps = 8;
constexpr int kAsmThreads = kAsmWarps * 32;
constexpr int kTilePad = 33;
constexpr size_t assemble_smem_bytes() { return (size_t)kAsmWarps * 32 * kTilePad * sizeof(double); }

// Potential-only term of Eq. 4.1: 12 FP64-pipe instructions (3 DADD + 3 DMUL + 6 DFMA).
__device__ __forceinline__ double phi_one(const double4 s, double q, double px, double py, double pz, double acc) {
  const double dx = __dsub_rn(px, s.x), dy = __dsub_rn(py, s.y), dz = __dsub_rn(pz, s.z);
  const double r2 = __fma_rn(dx, dx, __fma_rn(dy, dy, __dmul_rn(dz, dz)));
  return __fma_rn(q, rsqrt_f64(r2), acc);
}

__global__ void __launch_bounds__(kAsmThreads, 2) assemble_kernel(const __grid_constant__ AssembleParams p) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int64_t ct = (int64_t)blockIdx.x * kAsmWarps + warp;  // column tile
  const int64_t j0 = ct * 32;
  if (j0 >= p.n) return;
  const int64_t r0 = (int64_t)blockIdx.y * 32;  // first row of the tile, relative to row0
  double* tile = reinterpret_cast<double*>(smem_raw) + (size_t)warp * 32 * kTilePad;

  // rows: field points = centroids
  const int64_t nrow_here = min((int64_t)32, p.nrows - r0);
  const int64_t irow = p.row0 + r0 + min((int64_t)lane, nrow_here - 1);
  const double4 ci = p.cenL[irow];
  const double px = ci.x, py = ci.y, pz = ci.z;
  const double lox = warp_min(px), hix = warp_max(px), loy = warp_min(py), hiy = warp_max(py), loz = warp_min(pz),
               hiz = warp_max(pz);
  const double cx = 0.5 * (lox + hix), cy = 0.5 * (loy + hiy), cz = 0.5 * (loz + hiz);
  const double rho = sqrt(warp_max((px - cx) * (px - cx) + (py - cy) * (py - cy) + (pz - cz) * (pz - cz)));
  const double mag = fmax(fmax(fabs(cx), fabs(cy)), fabs(cz)) + rho;

  // columns: classify element j0 + lane against the row tile's bounding sphere
  int lnear = 0, lfar = 0, tcol = 0;
  double4 cj = make_double4(0, 0, 0, 1);
  if (j0 + lane < p.n) {
    cj = p.cenL[j0 + lane];
    tcol = p.type[j0 + lane];
    const double dx = cx - cj.x, dy = cy - cj.y, dz = cz - cj.z;
    const double Dc = sqrt(dx * dx + dy * dy + dz * dz);
    const double slack = 1e-9 * (Dc + rho) + 1e-12 * (mag + fmax(fmax(fabs(cj.x), fabs(cj.y)), fabs(cj.z)));
    const double Dhi = Dc + rho + slack, Dlo = fmax(Dc - rho - slack, 0.0);
    lfar = p.pol.map[want_level(Dhi * Dhi, cj.w, p.pol.dr[tcol])];
    lnear = p.pol.map[want_level(Dlo * Dlo, cj.w, p.pol.dr[tcol])];
    // the analytic formula is never an "upgrade" (see eval_adaptive_kernel): a tile straddling
    // the analytic limit keeps the exact per-pair choice
    if (p.pol.allow_upgrade && lnear != 5) lfar = lnear;
  }

  unsigned long long n_inter = 0, n_ana = 0;
  const int ncol_here = (int)min((int64_t)32, p.n - j0);
  for (int jj = 0; jj < ncol_here; ++jj) {
    const int64_t j = j0 + jj;
    const int ln = __shfl_sync(kFullMask, lnear, jj), lf = __shfl_sync(kFullMask, lfar, jj);
    const int t = __shfl_sync(kFullMask, tcol, jj);
    double val = 0.0;
    int lev = ln;
    if (ln != lf) {  // exact per-pair choice
      const double ex = __shfl_sync(kFullMask, cj.x, jj), ey = __shfl_sync(kFullMask, cj.y, jj),
                   ez = __shfl_sync(kFullMask, cj.z, jj), Lj = __shfl_sync(kFullMask, cj.w, jj);
      const double dx = __dsub_rn(px, ex), dy = __dsub_rn(py, ey), dz = __dsub_rn(pz, ez);
      const double D2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
      lev = p.pol.map[want_level(D2, Lj, p.pol.dr[t])];
    }
    for (int l = lf; l <= ln; ++l) {  // lf <= ln: the near end needs the more accurate level
      const bool take = (lev == l);
      if (!__any_sync(kFullMask, take)) continue;
      if (l == 5) {
        if (take) {
          Vec3 V[4];
          const int nv = load_polygon(p.type, p.verts, j, V);
          double ip;
          Vec3 ie;
          analytic_integrals<false>(V, nv, Vec3{px, py, pz}, ip, ie);
          val = ip;
          if (lane < nrow_here) n_ana += 1;
        }
      } else {
        const int N = rule_npts(t, l);
        const double4* src = p.lvl_pts[l] + j * p.stride[l];
        double acc = 0.0;
#pragma unroll 4
        for (int i = 0; i < N; ++i) {
          const double4 s = ldg4(src + i);
          acc = phi_one(s, s.w, px, py, pz, acc);
        }
        if (take) {
          val = acc;
          if (lane < nrow_here) n_inter += N;
        }
      }
    }
    tile[lane * kTilePad + jj] = p.k * val;
  }
  __syncwarp();
  for (int rr = 0; rr < (int)nrow_here; ++rr) {
    if (lane < ncol_here) p.out[(r0 + rr) * p.ld + j0 + lane] = tile[rr * kTilePad + lane];
  }
  if (p.counters) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      n_inter += __shfl_xor_sync(kFullMask, n_inter, o);
      n_ana += __shfl_xor_sync(kFullMask, n_ana, o);
    }
    if (lane == 0) {
      atomicAdd(p.counters, n_inter);
      if (n_ana) atomicAdd(p.counters + 1, n_ana);
    }
  }
}

}  // namespace bemcub
