// Steps a2 + a3 + a4 of the hot path: the point-charge sum of Eq. 4.1
// at many field points, with either one fixed rule or the distance-ratio
// choice of Sec. 4 (L159).
//
// Execution model (both kernels): PERSISTENT grid, one CTA of 12 warps per SM, every WARP an
// autonomous worker that pulls work items from a global atomic queue until it is empty.  One item
// = (tile of 32*R field points) x (one contiguous range of elements, a "split").  The warp keeps
// its 32*R field points in registers (lane l holds points tile*32R + r*32 + l, r < R) and streams
// the packed (x,y,z,q) point records of the split through its private double-buffered shared-memory
// window, filled by 1-D bulk TMA copies (cp.async.bulk -> UBLKCP) that complete on a per-warp
// mbarrier.  There is no __syncthreads anywhere: warps never wait for each other, so a tile that
// needs high-order rules (more points) delays nobody, and the tail of the launch is at most one
// item long.  The inner loop reads one point with two broadcast LDS.128 and applies it to the R
// field points of each lane: 18 FP64-pipe instructions per point-charge interaction
// (4 DADD + 6 DMUL + 8 DFMA = 26 flop) plus one MUFU.RSQ64H.  R = 4 gives four independent
// dependency chains per lane; with 3 warps per scheduler that nearly saturates the FP64 pipe
// (bare loop, field points from memory: 96 % of the DFMA-only issue rate at R = 4, 94 % at R = 2,
// 88 % at R = 1; what is missing is register-file bandwidth, not issue slots).
//
// Adaptive kernel: per batch of 32 elements each lane classifies ONE element against the bounding
// sphere of the warp's field points (conservative in both directions), so the rule of an element
// is warp-uniform: elements whose whole tile falls in one distance-ratio band are streamed at that
// level (consecutive elements merge into one bulk copy); an element whose tile straddles a band
// limit is either evaluated with the more accurate rule (allow_upgrade) or pair by pair with the
// exact per-pair choice; elements below the analytic limit go through analytic_integrals().
#pragma once
#include <math_constants.h>
#include <type_traits>
#include "analytic.cuh"
#include "device_utils.cuh"
#include "kernels_pre.cuh"

namespace bemcub {

constexpr int kWarpsPerCta = 12;  // 1 CTA per SM, 3 warps per scheduler, <= 168 registers per thread (16 warps at 128 registers spill in the loop: 0.6 % slower in round 2, 3 % in round 1)
constexpr int kThreads = kWarpsPerCta * 32;
constexpr int kBuf = 128;  // points per stage of a warp's window
constexpr int kStages = 2;
// source points per trip of the R = 4 loops (two per trip was measured on config 4 at full size: 0.3 % slower)
constexpr int kUnrollR4 = 1;

// Per-warp bookkeeping kept in shared memory (not registers): bounding sphere of the current tile
// and the interaction tallies.
struct WarpScratch {
  double cx, cy, cz, rho, mag;
  unsigned long long n_inter, n_ana;
  int nvalid, pad;
};

// shared memory of one CTA: [warps][stages][kBuf] points | [warps][stages] mbarriers | [warps] scratch
template <typename T>
constexpr size_t eval_smem_bytes() {
  return (size_t)kWarpsPerCta * kStages * kBuf * sizeof(typename Point4<T>::type) + (size_t)kWarpsPerCta * kStages * 8 +
         (size_t)kWarpsPerCta * sizeof(WarpScratch);
}

// Next work item of the persistent loop (lane 0 pulls, the warp shares it).
__device__ __forceinline__ int64_t next_item(unsigned long long* queue, int lane) {
  unsigned long long it = 0;
  if (lane == 0) it = atomicAdd(queue, 1ull);
  return (int64_t)__shfl_sync(kFullMask, it, 0);
}

// What a kernel accumulates per field point: Phi and E (Eq. 4.1), Phi, E and the field gradient
// (L273), or the potential alone (the mat-vec of a BEM solve, L34; any call without out_E).
constexpr int kModePhiE = 0, kModeGrad = 1, kModePhi = 2;

// Running sums of one lane.  kModeGrad adds the six sums the field gradient needs:
// sg = sum q/r^3 and s_ab = sum 3 q d_a d_b / r^5, from which G_ab = k (delta_ab sg - s_ab).
template <typename T, int R, int MODE = kModePhiE>
struct Accum {
  static constexpr int RG = (MODE == kModeGrad) ? R : 1;
  T phi[R], ex[R], ey[R], ez[R];
  T sg[RG], sxx[RG], syy[RG], sxy[RG], sxz[RG], syz[RG];
  __device__ __forceinline__ void zero() {
#pragma unroll
    for (int r = 0; r < R; ++r) phi[r] = ex[r] = ey[r] = ez[r] = (T)0;
#pragma unroll
    for (int r = 0; r < RG; ++r) sg[r] = sxx[r] = syy[r] = sxy[r] = sxz[r] = syz[r] = (T)0;
  }
};

// One point charge (sx,sy,sz,q) seen from one field point: Eq. 4.1 term.
__device__ __forceinline__ void interact_one(double sx, double sy, double sz, double q, double px, double py, double pz,
                                             double& phi, double& ex, double& ey, double& ez, double c375) {
  const double dx = __dsub_rn(px, sx), dy = __dsub_rn(py, sy), dz = __dsub_rn(pz, sz);
  const double yz = __fma_rn(dy, dy, __dmul_rn(dz, dz));
  const double r2 = __fma_rn(dx, dx, yz);
  const double y = rsqrt_f64(r2, yz, c375);  // 1/|P-Q_i|: "one square root and one division" (L46)
  const double qy = __dmul_rn(q, y);
  phi = __dadd_rn(phi, qy);
  const double y2 = __dmul_rn(y, y);
  const double g = __dmul_rn(qy, y2);  // q / r^3
  ex = __fma_rn(dx, g, ex);
  ey = __fma_rn(dy, g, ey);
  ez = __fma_rn(dz, g, ez);
}
// Potential only: 12 FP64-pipe instructions (3 DADD + 3 DMUL + 6 DFMA).
__device__ __forceinline__ void interact_one_phi(double sx, double sy, double sz, double q, double px, double py, double pz,
                                                 double& phi, double c375) {
  const double dx = __dsub_rn(px, sx), dy = __dsub_rn(py, sy), dz = __dsub_rn(pz, sz);
  const double r2 = __fma_rn(dx, dx, __fma_rn(dy, dy, __dmul_rn(dz, dz)));
  phi = __fma_rn(q, rsqrt_f64(r2, dz, c375), phi);
}
__device__ __forceinline__ void interact_one_phi(float sx, float sy, float sz, float q, float px, float py, float pz, float& phi,
                                                 double) {
  const float dx = px - sx, dy = py - sy, dz = pz - sz;
  phi = fmaf(q, rsqrt_f32(fmaf(dx, dx, fmaf(dy, dy, dz * dz))), phi);
}
// The same term plus its derivative sums: 10 more FP64 instructions (4 DMUL + 1 DADD + 5 DFMA).
// s_zz is never formed: h r^2 = 3 g makes the gradient traceless, G_zz = -(G_xx + G_yy).
__device__ __forceinline__ void interact_one_grad(double sx, double sy, double sz, double q, double px, double py, double pz,
                                                  double& phi, double& ex, double& ey, double& ez, double& sg, double& sxx,
                                                  double& syy, double& sxy, double& sxz, double& syz, double c375) {
  const double dx = __dsub_rn(px, sx), dy = __dsub_rn(py, sy), dz = __dsub_rn(pz, sz);
  const double yz = __fma_rn(dy, dy, __dmul_rn(dz, dz));
  const double r2 = __fma_rn(dx, dx, yz);
  const double y = rsqrt_f64(r2, yz, c375);
  const double qy = __dmul_rn(q, y);
  phi = __dadd_rn(phi, qy);
  const double y2 = __dmul_rn(y, y);
  const double g = __dmul_rn(qy, y2);  // q / r^3
  ex = __fma_rn(dx, g, ex);
  ey = __fma_rn(dy, g, ey);
  ez = __fma_rn(dz, g, ez);
  const double h = __dmul_rn(g, __dmul_rn(3.0, y2));  // 3 q / r^5
  const double hx = __dmul_rn(h, dx), hy = __dmul_rn(h, dy);
  sg = __dadd_rn(sg, g);
  sxx = __fma_rn(hx, dx, sxx);
  syy = __fma_rn(hy, dy, syy);
  sxy = __fma_rn(hx, dy, sxy);
  sxz = __fma_rn(hx, dz, sxz);
  syz = __fma_rn(hy, dz, syz);
}
__device__ __forceinline__ void interact_one(float sx, float sy, float sz, float q, float px, float py, float pz,
                                             float& phi, float& ex, float& ey, float& ez, double) {
  const float dx = px - sx, dy = py - sy, dz = pz - sz;
  const float r2 = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
  const float y = rsqrt_f32(r2);
  const float qy = q * y;
  phi += qy;
  const float g = qy * (y * y);
  ex = fmaf(dx, g, ex);
  ey = fmaf(dy, g, ey);
  ez = fmaf(dz, g, ez);
}

template <typename T, int R, int MODE, typename P4>
__device__ __forceinline__ void interact(const P4 s, const T (&px)[R], const T (&py)[R], const T (&pz)[R],
                                         Accum<T, R, MODE>& a, double c375) {
#pragma unroll
  for (int r = 0; r < R; ++r) {
    if constexpr (MODE == kModeGrad)
      interact_one_grad(s.x, s.y, s.z, s.w, px[r], py[r], pz[r], a.phi[r], a.ex[r], a.ey[r], a.ez[r], a.sg[r], a.sxx[r],
                        a.syy[r], a.sxy[r], a.sxz[r], a.syz[r], c375);
    else if constexpr (MODE == kModePhi)
      interact_one_phi(s.x, s.y, s.z, s.w, px[r], py[r], pz[r], a.phi[r], c375);
    else
      interact_one(s.x, s.y, s.z, s.w, px[r], py[r], pz[r], a.phi[r], a.ex[r], a.ey[r], a.ez[r], c375);
  }
}

// All `cnt` points of a filled window applied to the warp's field points, U points per trip so
// that a lane always has >= 4 independent interaction chains in flight.
template <typename T, int R, int MODE, typename P4>
__device__ __forceinline__ void consume(const P4* __restrict__ buf, int cnt, const T (&px)[R], const T (&py)[R],
                                        const T (&pz)[R], Accum<T, R, MODE>& a) {
  constexpr int U = R >= 4 ? kUnrollR4 : (R >= 2 ? 2 : 4);
  const double c375 = c_three_eighths;
  int i = 0;
#pragma unroll 1
  for (; i + U <= cnt; i += U) {
    P4 s[U];
#pragma unroll
    for (int u = 0; u < U; ++u) s[u] = buf[i + u];
#pragma unroll
    for (int u = 0; u < U; ++u) interact<T, R, MODE>(s[u], px, py, pz, a, c375);
  }
#pragma unroll 1
  for (; i < cnt; ++i) interact<T, R, MODE>(buf[i], px, py, pz, a, c375);
}

// FP64: the window's sum goes straight into the running totals.  FP32: the window (<= kBuf
// terms) is summed in FP32 and the block sum is added to FP64 totals (reading 11).
template <int R, int MODE>
__device__ __forceinline__ void consume_into(const double4* buf, int cnt, const double (&px)[R], const double (&py)[R],
                                             const double (&pz)[R], Accum<double, R, MODE>& tot) {
  consume<double, R, MODE>(buf, cnt, px, py, pz, tot);
}
template <int R, int MODE>
__device__ __forceinline__ void consume_into(const float4* buf, int cnt, const float (&px)[R], const float (&py)[R],
                                             const float (&pz)[R], Accum<double, R, MODE>& tot) {
  static_assert(MODE != kModeGrad, "the field gradient is FP64 only");
  Accum<float, R, MODE> a;
  a.zero();
  consume<float, R, MODE>(buf, cnt, px, py, pz, a);
#pragma unroll
  for (int r = 0; r < R; ++r) {
    tot.phi[r] += (double)a.phi[r];
    tot.ex[r] += (double)a.ex[r];
    tot.ey[r] += (double)a.ey[r];
    tot.ez[r] += (double)a.ez[r];
  }
}

__device__ __forceinline__ double4 ldg_point(const double4* p) { return ldg4(p); }
__device__ __forceinline__ float4 ldg_point(const float4* p) { return __ldg(p); }

template <typename T, int R>
__device__ __forceinline__ void load_field_points(const double* __restrict__ field, int64_t m, int64_t tile, int lane,
                                                  T (&px)[R], T (&py)[R], T (&pz)[R]) {
#pragma unroll
  for (int r = 0; r < R; ++r) {
    int64_t j = tile * (32 * R) + r * 32 + lane;
    if (j >= m) j = m - 1;  // clamped duplicates compute harmlessly and are never stored
    px[r] = (T)field[3 * j];
    py[r] = (T)field[3 * j + 1];
    pz[r] = (T)field[3 * j + 2];
  }
}

// partial_g (gradient mode only): [m][6] = sg, sxx, syy, sxy, sxz, syz of this split
template <int R, int MODE>
__device__ __forceinline__ void store_partial(double4* __restrict__ partial, double* __restrict__ partial_g, int64_t m,
                                              int64_t tile, int lane, const Accum<double, R, MODE>& tot) {
#pragma unroll
  for (int r = 0; r < R; ++r) {
    const int64_t j = tile * (32 * R) + r * 32 + lane;
    if (j < m) {
      partial[j] = make_double4(tot.phi[r], tot.ex[r], tot.ey[r], tot.ez[r]);
      if constexpr (MODE == kModeGrad) {
        double2* g = reinterpret_cast<double2*>(partial_g + 6 * j);
        g[0] = make_double2(tot.sg[r], tot.sxx[r]);
        g[1] = make_double2(tot.syy[r], tot.sxy[r]);
        g[2] = make_double2(tot.sxz[r], tot.syz[r]);
      }
    }
  }
}

// ------------------------------------------------------------------------------------------------
// Shared-memory carve-up of the calling warp.
template <typename P4>
struct WarpSmem {
  P4* win;           // [kStages][kBuf]
  uint32_t win0;     // shared-space address of win
  uint32_t bar0;     // shared-space address of the first of kStages mbarriers (8 bytes apart)
  WarpScratch* scr;
};
template <typename P4>
__device__ __forceinline__ WarpSmem<P4> warp_smem(unsigned char* smem_raw, int warp, int lane) {
  WarpSmem<P4> w;
  w.win = reinterpret_cast<P4*>(smem_raw) + (size_t)warp * kStages * kBuf;
  unsigned char* after = smem_raw + (size_t)kWarpsPerCta * kStages * kBuf * sizeof(P4);
  uint64_t* bars = reinterpret_cast<uint64_t*>(after) + warp * kStages;
  w.scr = reinterpret_cast<WarpScratch*>(after + (size_t)kWarpsPerCta * kStages * 8) + warp;
  w.win0 = smem_u32(w.win);
  w.bar0 = smem_u32(bars);
  if (lane == 0) {
    mbar_init(w.bar0, 1);
    mbar_init(w.bar0 + 8, 1);
    mbar_fence_init();
    w.scr->n_inter = 0;
    w.scr->n_ana = 0;
  }
  __syncwarp();
  return w;
}

// Packing of a classified 32-element batch into a warp's window (adaptive evaluation and matrix fill
// share it).  Lane l holds element l of the batch: cnt points (0 = not streamed) of level lvl, pre =
// exclusive prefix of cnt, total = its sum.  Starting at lane `cursor`, the next stage takes whole
// elements while they fit into kBuf points; consecutive elements of one level whose records are
// adjacent in memory (cnt == stride of the level) are merged into one bulk copy, issued by the run's
// first lane.
struct StagePlan {
  int base;      // pre of the first lane of the stage
  int next;      // first lane that does not fit (32 = batch exhausted): the next cursor
  int nstage;    // points of the stage
  int run_end;   // this lane heads a copy run: pre of the lane after the run
  bool inc;      // this lane's element is in the stage
  bool head;     // ... and starts a copy run
  unsigned incmask;
};
__device__ __forceinline__ StagePlan plan_stage(int cursor, int lane, int cnt, int pre, int total, int lvl, const int (&stride)[5]) {
  StagePlan s;
  s.base = __shfl_sync(kFullMask, pre, cursor);
  const bool after = lane >= cursor;
  const unsigned nofit = __ballot_sync(kFullMask, after && (pre + cnt - s.base > kBuf));
  s.next = nofit ? (__ffs(nofit) - 1) : 32;
  const int pre_next = __shfl_sync(kFullMask, pre, s.next & 31);
  const int endp = (s.next < 32) ? pre_next : total;
  s.nstage = endp - s.base;
  s.inc = after && lane < s.next && cnt > 0;
  const int prev_cnt = __shfl_up_sync(kFullMask, cnt, 1);
  const int prev_lvl = __shfl_up_sync(kFullMask, lvl, 1);
  // a lane continues its predecessor's copy if that one ends exactly where this one starts
  const bool cont = s.inc && lane > cursor && lvl >= 0 && prev_cnt > 0 && prev_lvl == lvl && prev_cnt == stride[lvl];
  s.incmask = __ballot_sync(kFullMask, s.inc);
  s.head = s.inc && !cont;
  const unsigned heads = __ballot_sync(kFullMask, s.head);
  const unsigned higher = heads & ~((2u << lane) - 1u);
  const int h2 = higher ? (__ffs(higher) - 1) : 32;
  const int pre_h2 = __shfl_sync(kFullMask, pre, h2 & 31);
  s.run_end = (h2 < 32) ? pre_h2 : endp;
  return s;
}

struct FixedParams {
  const void* pts;          // Point4<T>[npts], one rule level
  int64_t npts;             // n * stride
  int64_t pts_per_split;    // elements per split * stride
  const double* field;      // [m][3]
  int64_t m;
  double4* partial;         // [nsplit][split_stride]
  double* partial_g;        // [nsplit][split_stride][6], gradient sums (gradient kernels only)
  int64_t split_stride;
  int64_t ntiles;           // ceil(m / (32 R))
  int64_t nitems;           // ntiles * nsplit; item = split * ntiles + tile
  unsigned long long* queue;  // work-item counter, zeroed before the launch
  unsigned long long* counters;  // [4], [5]: cycles and nanoseconds of the launch (KernelClock)
};

template <typename T, int R, int MODE = kModePhiE>
__global__ void __launch_bounds__(kThreads, 1) eval_fixed_kernel(const __grid_constant__ FixedParams p) {
  typedef typename Point4<T>::type P4;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const WarpSmem<P4> ws = warp_smem<P4>(smem_raw, warp, lane);
  const P4* src = reinterpret_cast<const P4*>(p.pts);
  uint32_t phases = 0;  // parity of each stage's mbarrier, carried across items
  KernelClock clk;
  clk.begin();

  for (;;) {
    const int64_t item = next_item(p.queue, lane);
    if (item >= p.nitems) break;
    const int64_t split = item / p.ntiles, tile = item - split * p.ntiles;

    T px[R], py[R], pz[R];
    load_field_points<T, R>(p.field, p.m, tile, lane, px, py, pz);
    const int64_t q0 = split * p.pts_per_split;
    const int64_t q1 = min(p.npts, q0 + p.pts_per_split);
    const int64_t nchunks = (q1 - q0 + kBuf - 1) / kBuf;

    Accum<double, R, MODE> tot;
    tot.zero();
    auto fill = [&](int64_t c, int stage) {
      if (lane == 0) {
        const int64_t a = q0 + c * kBuf;
        const uint32_t bytes = (uint32_t)(min((int64_t)kBuf, q1 - a) * sizeof(P4));
        mbar_arrive_expect_tx(ws.bar0 + 8 * stage, bytes);
        tma_load_1d(ws.win0 + stage * (uint32_t)(kBuf * sizeof(P4)), src + a, bytes, ws.bar0 + 8 * stage);
      }
    };
    if (nchunks > 0) fill(0, 0);
    for (int64_t c = 0; c < nchunks; ++c) {
      const int stage = (int)(c & 1);
      if (c + 1 < nchunks) fill(c + 1, stage ^ 1);
      mbar_wait(ws.bar0 + 8 * stage, (phases >> stage) & 1u);
      phases ^= 1u << stage;
      const int cnt = (int)min((int64_t)kBuf, q1 - (q0 + c * kBuf));
      consume_into<R, MODE>(ws.win + stage * kBuf, cnt, px, py, pz, tot);
      __syncwarp();  // every lane is done with this stage before it is refilled
    }
    store_partial<R, MODE>(p.partial + split * p.split_stride, (MODE == kModeGrad) ? p.partial_g + split * p.split_stride * 6 : nullptr, p.m,
                           tile, lane, tot);
  }
  clk.end(p.counters);
}

// ------------------------------------------------------------------------------------------------
// Distance-ratio policy on the device.  map[want] = level actually used for a wanted level
// (use_levels_mask applied on the host).
struct PolicyDev {
  double dr[2][5];
  int map[6];
  int allow_upgrade;
};

// Band of a squared distance: the smallest b with D^2 < (dr[b] L)^2 gives level 5-b (b = 0 is the
// analytic branch); none gives level 0 (N = 4).  Lower-inclusive bands (reading 8).
__device__ __forceinline__ int want_level(double D2, double L, const double* dr5) {
  int want = 0;
#pragma unroll
  for (int b = 4; b >= 0; --b) {
    const double thr = __dmul_rn(dr5[b], L);
    if (D2 < __dmul_rn(thr, thr)) want = 5 - b;
  }
  return want;
}

__device__ __forceinline__ int rule_npts(int type, int level) {
  return type == 0 ? (c_tri_off[level + 1] - c_tri_off[level]) : (c_rect_off[level + 1] - c_rect_off[level]);
}

struct AdaptiveParams {
  const void* lvl_pts[5];  // expanded points per level (Point4<T> records), may be null for disabled levels
  int stride[5];
  const double4* cenL;
  const uint8_t* type;
  const double* verts;
  const double* sigma;
  int64_t n;
  int64_t elems_per_split;
  PolicyDev pol;
  const double* field;
  int64_t m;
  double4* partial;
  double* partial_g;  // gradient sums (gradient kernels only)
  int64_t split_stride;
  int64_t ntiles;
  int64_t nitems;
  unsigned long long* queue;
  unsigned long long* counters;  // [0] point-charge interactions, [1] analytic pairs
};

// Field points of the warp's current tile.
template <int R>
struct WarpTile {
  double px[R], py[R], pz[R];
  int64_t first;  // index of the tile's first field point
  int64_t m;
  __device__ __forceinline__ bool ok(int r, int lane) const { return first + r * 32 + lane < m; }
};

__device__ __forceinline__ int warp_sum(int v) { return __reduce_add_sync(kFullMask, v); }

// Element `e` evaluated analytically at the field points of the tile selected by `take` (a4).
template <int R, int MODE>
__device__ __forceinline__ void analytic_element(const AdaptiveParams& p, int64_t e, const WarpTile<R>& w, const bool (&take)[R],
                                              Accum<double, R, MODE>& tot) {
  Vec3 V[4];
  const int nv = load_polygon(p.type, p.verts, e, V);
  const double sg = __ldg(p.sigma + e);
#pragma unroll
  for (int r = 0; r < R; ++r) {
    if (!take[r]) continue;
    double ip;
    Vec3 ie;
    if constexpr (MODE == kModePhi) {
      analytic_integrals<false>(V, nv, Vec3{w.px[r], w.py[r], w.pz[r]}, ip, ie);
      tot.phi[r] += sg * ip;
    } else {
      analytic_integrals<true>(V, nv, Vec3{w.px[r], w.py[r], w.pz[r]}, ip, ie);
      tot.phi[r] += sg * ip;
      tot.ex[r] += sg * ie.x;
      tot.ey[r] += sg * ie.y;
      tot.ez[r] += sg * ie.z;
    }
  }
}

// Element `e` with the exact per-pair rule choice (tile straddles a band limit and the policy
// does not allow, or the analytic limit forbids, an upgrade).  T = float: points and interaction
// arithmetic in FP32 (one element's sum: at most 33 terms), added to the FP64 totals.
template <typename T, int R, int MODE>
__device__ __forceinline__ void mixed_element(const AdaptiveParams& p, int64_t e, const WarpTile<R>& w, const T (&qx)[R],
                                              const T (&qy)[R], const T (&qz)[R], int lane, Accum<double, R, MODE>& tot,
                                              WarpScratch* scr) {
  typedef typename Point4<T>::type P4;
  const double4 c = ldg4(p.cenL + e);
  const int t = __ldg(p.type + e);
  int lev[R];
#pragma unroll
  for (int r = 0; r < R; ++r) {
    const double dx = __dsub_rn(w.px[r], c.x), dy = __dsub_rn(w.py[r], c.y), dz = __dsub_rn(w.pz[r], c.z);
    const double D2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
    lev[r] = p.pol.map[want_level(D2, c.w, p.pol.dr[t])];
  }
  for (int l = 0; l <= 5; ++l) {
    bool take[R];
    bool any = false;
    int mine = 0;
#pragma unroll
    for (int r = 0; r < R; ++r) {
      take[r] = (lev[r] == l);
      any |= take[r];
      mine += (take[r] && w.ok(r, lane)) ? 1 : 0;
    }
    if (!__any_sync(kFullMask, any)) continue;
    const int all = warp_sum(mine);
    if (l == 5) {
      analytic_element<R, MODE>(p, e, w, take, tot);  // never reached in gradient mode: the host rejects such policies
      if (lane == 0) scr->n_ana += (unsigned long long)all;
    } else {
      const int N = rule_npts(t, l);
      const P4* src = reinterpret_cast<const P4*>(p.lvl_pts[l]) + e * p.stride[l];
      // The level's sum is formed for every field point of the lane and then SELECTED, not masked
      // by a zero charge: a field point that does not take this level may sit exactly on one of its
      // nodes (an element's own centroid is a node of the 7- and 19-point rules), and 0 * inf = NaN.
      Accum<T, R, MODE> part;
      part.zero();
      P4 s = ldg_point(src);
      const double c375 = c_three_eighths;
#pragma unroll 1
      for (int i = 0; i < N; ++i) {
        const P4 nxt = ldg_point(src + min(i + 1, N - 1));  // prefetch: hides the global-load latency
        interact<T, R, MODE>(s, qx, qy, qz, part, c375);
        s = nxt;
      }
#pragma unroll
      for (int r = 0; r < R; ++r) {
        if (!take[r]) continue;
        tot.phi[r] += (double)part.phi[r];
        if constexpr (MODE != kModePhi) {
          tot.ex[r] += (double)part.ex[r];
          tot.ey[r] += (double)part.ey[r];
          tot.ez[r] += (double)part.ez[r];
        }
        if constexpr (MODE == kModeGrad) {
          tot.sg[r] += part.sg[r];
          tot.sxx[r] += part.sxx[r];
          tot.syy[r] += part.syy[r];
          tot.sxy[r] += part.sxy[r];
          tot.sxz[r] += part.sxz[r];
          tot.syz[r] += part.syz[r];
        }
      }
      if (lane == 0) scr->n_inter += (unsigned long long)all * N;
    }
  }
}

// T = double: the FP64 path.  T = float: the points, the field points of the interaction and its
// arithmetic are FP32 (window sums of <= kBuf terms, added to FP64 totals); the rule choice and the
// analytic branch stay FP64.
template <typename T, int R, int MODE = kModePhiE>
__global__ void __launch_bounds__(kThreads, 1) eval_adaptive_kernel(const __grid_constant__ AdaptiveParams p) {
  typedef typename Point4<T>::type P4;
  static_assert(sizeof(T) == 8 || MODE != kModeGrad, "the field gradient is FP64 only");
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const WarpSmem<P4> ws = warp_smem<P4>(smem_raw, warp, lane);
  WarpScratch* const scr = ws.scr;
  uint32_t phases = 0;
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
    float fx[sizeof(T) == 8 ? 1 : R], fy[sizeof(T) == 8 ? 1 : R], fz[sizeof(T) == 8 ? 1 : R];  // FP32 path: narrowed copies
    if constexpr (sizeof(T) == 4) {
#pragma unroll
      for (int r = 0; r < R; ++r) {
        fx[r] = (float)w.px[r]; fy[r] = (float)w.py[r]; fz[r] = (float)w.pz[r];
      }
    }
    {  // bounding sphere of the tile (clamped duplicates lie inside it by construction).  Points
       // with a non-finite coordinate are left out: their own result is NaN whatever the rule, and
       // they must not spoil the rule choice of the other points of the tile.
      // (fmin / fmax / warp_min / warp_max return the other operand when one is NaN, so a point is
      // left out by turning its coordinates into NaN for this computation only)
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
      const bool any_fin = lox <= hix;  // false if every point of the tile is non-finite (NaN compares false)
      const double cx = any_fin ? 0.5 * (lox + hix) : 0.0, cy = any_fin ? 0.5 * (loy + hiy) : 0.0,
                   cz = any_fin ? 0.5 * (loz + hiz) : 0.0;
      double d2 = 0.0;
#pragma unroll
      for (int r = 0; r < R; ++r) {
        const double dx = w.px[r] - cx, dy = w.py[r] - cy, dz = w.pz[r] - cz;
        const double t = dx * dx + dy * dy + dz * dz;
        d2 = fmax(d2, t <= 1e300 ? t : 0.0);  // a non-finite point (t = NaN or inf) does not widen the sphere
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

    // state of the current 32-element batch: lane l holds element batch0 + l.  (Parking it in shared
    // memory between two produce() calls was measured: no gain at scale 0.25, 3 % slower at full size.)
    int64_t batch_next = e_begin;
    int cnt = 0, pre = 0, total = 0, lvl = 0, cursor = 32;
    const P4* src = nullptr;

    // Fills `stage` with the next round of whole elements; returns the number of points (0 = done).
    auto produce = [&](int stage) -> int {
      for (;;) {
        if (cursor < 32) {
          const StagePlan sp = plan_stage(cursor, lane, cnt, pre, total, lvl, p.stride);
          const int nstage = sp.nstage;
          cursor = sp.next;
          if (nstage == 0) continue;
          if (lane == 0) mbar_arrive_expect_tx(ws.bar0 + 8 * stage, (uint32_t)(nstage * sizeof(P4)));
          __syncwarp();
          if (sp.head)
            tma_load_1d(ws.win0 + (uint32_t)((stage * kBuf + (pre - sp.base)) * sizeof(P4)), src,
                        (uint32_t)((sp.run_end - pre) * sizeof(P4)), ws.bar0 + 8 * stage);
          if (lane == 0) scr->n_inter += (unsigned long long)nstage * scr->nvalid;
          return nstage;
        }
        if (batch_next >= e_end) return 0;
        // ---- a2: classify 32 elements, one per lane, against the tile's bounding sphere
        const int64_t batch0 = batch_next;
        const int64_t e = batch0 + lane;
        batch_next += 32;
        cnt = 0;
        lvl = -1;
        bool is_ana = false, is_mixed = false;
        if (e < e_end) {
          const double4 c = p.cenL[e];
          const int t = p.type[e];
          const double rho = scr->rho;
          const double dx = scr->cx - c.x, dy = scr->cy - c.y, dz = scr->cz - c.z;
          const double Dc = sqrt(dx * dx + dy * dy + dz * dz);
          const double slack =
              1e-9 * (Dc + rho) + 1e-12 * (scr->mag + fmax(fmax(fabs(c.x), fabs(c.y)), fabs(c.z)));
          const double Dhi = Dc + rho + slack;
          const double Dlo = fmax(Dc - rho - slack, 0.0);
          const int lfar = p.pol.map[want_level(Dhi * Dhi, c.w, p.pol.dr[t])];
          const int lnear = p.pol.map[want_level(Dlo * Dlo, c.w, p.pol.dr[t])];
          // A tile that straddles a band limit: per-pair choice, or (allow_upgrade) the more accurate
          // cubature rule for the whole tile.  The analytic formula is never an "upgrade": its
          // rounding error grows with the distance ratio (Figs. 2-4), so a tile that
          // straddles the analytic limit is always resolved pair by pair.
          if (lnear != lfar && (!p.pol.allow_upgrade || lnear == 5)) {
            is_mixed = true;
          } else {
            lvl = lnear;  // the more accurate end of the tile's range
            if (lvl == 5) {
              is_ana = true;
            } else {
              cnt = rule_npts(t, lvl);
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
          if constexpr (sizeof(T) == 8) mixed_element<double, R, MODE>(p, batch0 + l, w, w.px, w.py, w.pz, lane, tot, scr);
          else mixed_element<float, R, MODE>(p, batch0 + l, w, fx, fy, fz, lane, tot, scr);
        }
      }
    };

    // software pipeline with a single produce() call site: fill stage s^1, then consume stage s
    int cur = 0, stage = 1;
    for (;;) {
      const int nxt = produce(stage ^ 1);
      if (cur > 0) {
        mbar_wait(ws.bar0 + 8 * stage, (phases >> stage) & 1u);
        phases ^= 1u << stage;
        if constexpr (sizeof(T) == 8) consume_into<R, MODE>(ws.win + stage * kBuf, cur, w.px, w.py, w.pz, tot);
        else consume_into<R, MODE>(ws.win + stage * kBuf, cur, fx, fy, fz, tot);
        __syncwarp();
      }
      if (nxt == 0) break;
      stage ^= 1;
      cur = nxt;
    }
    store_partial<R, MODE>(p.partial + split * p.split_stride, (MODE == kModeGrad) ? p.partial_g + split * p.split_stride * 6 : nullptr, p.m,
                           tile, lane, tot);
  }

  __syncwarp();
  if (p.counters && lane == 0) {
    if (scr->n_inter) atomicAdd(p.counters, scr->n_inter);
    if (scr->n_ana) atomicAdd(p.counters + 1, scr->n_ana);
  }
  clk.end(p.counters);
}

// ------------------------------------------------------------------------------------------------
// Few field points (m <= kFewMaxM; particle tracking asks for the field at one point after the
// other): the roles are swapped.  Every THREAD owns elements (grid-stride), the
// field points of the pass (4; 1 or 2 if the call has no more) are shared by all lanes, every (element,
// point) pair gets its rule from its own distance ratio (the per-pair policy of L159, exactly), and the
// partial sums of the lanes are combined with warp shuffles, then across the warps of the CTA; the last
// CTA of a pass to finish adds the CTAs' sums in CTA order and applies k (step a6 inside the same launch).
// Such a call is bound by latency, not bandwidth: for one field point it reads 121 bytes per element
// (vertices, centroid, L, area, sigma) - 121 MB for 10^6 elements.  Round 2 measured where the 0.10 ms of
// such a call went: a pass of 4 with three clamped duplicates, one dependent load chain per thread, and a
// second launch whose single thread added 296 partial sums one L2 round trip after the other (45 us).
// Now: passes of 1 / 2 / 4 points, the next element's record loaded ahead of this one's arithmetic (1 / 2
// points: the registers allow it), the 7- and 12-point rules of such passes as straight-line code with the
// tables as constant operands (rule_point_ct), the sum over the CTAs inside the kernel: 0.041 ms for one
// point, 0.062 ms for two, 0.098 ms for four (config-4 mesh, 10^6 elements, sigma kept).
constexpr int kFewM = 4;        // field points per pass (grid.y); calls with 1 or 2 points run passes of 1 or 2
constexpr int kFewMaxM = 64;    // above this the tiled kernels win (10^6 elements: 1.4 ms at m = 64 either way; 2.9 ms tiled with a new sigma)
constexpr int kFewWarps = 8;

struct FewParams {
  const double4* cenL;
  const uint8_t* type;
  const double* verts;
  const double* sigma;
  int64_t n;
  PolicyDev pol;
  int rule;  // fixed level 0..4, or -1: per pair by distance ratio
  const double* field;
  int64_t m;
  double4* partial;  // [gridDim.x][m]
  unsigned long long* counters;
  const double* area;
  const double* sigma_v;  // linear density (may be null; then sigma is the constant density)
  unsigned* done;         // [gridDim.y] CTAs of each pass that have written their partial sums (zeroed before the launch)
  double k;               // 1/(4 pi eps0)
  double* out_phi;        // [m]
  double* out_E;          // [m][3] or null
};

__device__ __forceinline__ double warp_sum_f64(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(kFullMask, v, o);
  return v;
}

// The Gaussian points are computed on the fly from the vertices (the paper's own CPU variant, L218;
// Table 4 compares it with precomputed points): no preprocessing pass, 121 instead of 260 bytes
// read per element (reading precomputed points was measured 20 % slower here).
// (4 CTAs per SM at 64 registers were measured for the one-point kernel: spills, 127 instead of 76 us)
template <int MODE, int M>
__global__ void __launch_bounds__(kFewWarps * 32, 2) eval_few_kernel(const __grid_constant__ FewParams p) {
  constexpr int kFewM = M;  // field points of this pass
  __shared__ double red[kFewWarps][kFewM][4];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int64_t j0 = (int64_t)blockIdx.y * kFewM;
  const int mj = (int)min((int64_t)kFewM, p.m - j0);
  double px[kFewM], py[kFewM], pz[kFewM];
#pragma unroll
  for (int j = 0; j < kFewM; ++j) {
    const int64_t jj = j0 + min(j, mj - 1);  // clamped duplicates are never stored
    px[j] = p.field[3 * jj];
    py[j] = p.field[3 * jj + 1];
    pz[j] = p.field[3 * jj + 2];
  }
  Accum<double, kFewM, MODE> acc;
  acc.zero();
  const double c375 = c_three_eighths;
  unsigned long long n_inter = 0, n_ana = 0;

  // One element per thread and trip; the record of the next trip's element is loaded before this
  // trip's arithmetic starts (a call with few points is bound by the latency of these loads).
  struct Rec {
    double4 c;
    double v[9];
    double sg, ar;
    int t;
  };
  auto load_rec = [&](int64_t e, Rec& r) {
    r.c = p.cenL[e];
    r.t = p.type[e];
#pragma unroll
    for (int k = 0; k < 9; ++k) r.v[k] = __ldg(p.verts + 9 * e + k);
    r.sg = p.sigma ? __ldg(p.sigma + e) : 1.0;
    r.ar = __ldg(p.area + e);
  };
  const int64_t e_step = (int64_t)gridDim.x * blockDim.x;
  int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  constexpr bool kPrefetch = M <= 2;  // four points per pass: the second record does not fit the registers
  Rec nxt;
  if (kPrefetch && e < p.n) load_rec(e, nxt);
  for (; e < p.n; e += e_step) {
    Rec cur;
    if constexpr (kPrefetch) {
      cur = nxt;
      if (e + e_step < p.n) load_rec(e + e_step, nxt);
    } else {
      load_rec(e, cur);
    }
    const double4 c = cur.c;
    const int t = cur.t;
    const double (&v)[9] = cur.v;
    const double q = cur.sg * cur.ar;
    const double* sv = p.sigma_v ? p.sigma_v + 3 * e : nullptr;
    auto point = [&](int level, int i) -> double4 {
      double4 pt;
      rule_point(t, level, i, v, c, q, sv, pt);
      return pt;
    };
    int lev[kFewM];
    bool same = true;
#pragma unroll
    for (int j = 0; j < kFewM; ++j) {
      if (p.rule >= 0) {
        lev[j] = p.rule;
      } else {
        const double dx = __dsub_rn(px[j], c.x), dy = __dsub_rn(py[j], c.y), dz = __dsub_rn(pz[j], c.z);
        const double D2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
        lev[j] = p.pol.map[want_level(D2, c.w, p.pol.dr[t])];
      }
      same &= lev[j] == lev[0];
    }
    if (same && lev[0] != 5) {  // the usual case: one rule for all points of the pass
      const int N = rule_npts(t, lev[0]);
      // the 7- and 12-point rules (most pairs of a mesh seen from a distance, L181) with the tables as
      // constant operands of fully unrolled code; any other rule through the general rule_point()
      auto unrolled = [&](auto tt, auto ll) {
        constexpr int T = decltype(tt)::value, L = decltype(ll)::value;
        constexpr int NN = (T == 0 ? kTriOffCt[L + 1] - kTriOffCt[L] : kRectOffCt[L + 1] - kRectOffCt[L]);
#pragma unroll
        for (int i = 0; i < NN; ++i) {
          double4 pt;
          rule_point_ct<T, L>(i, v, c, q, sv, pt);
          interact<double, kFewM, MODE>(pt, px, py, pz, acc, c375);
        }
      };
      using std::integral_constant;
      // (four points per pass: the straight-line code of 28 - 48 interactions was measured 12 - 22 % slower
      // than the loop - registers and instruction cache - so only passes of one or two points take it)
      constexpr bool kUnrolled = M <= 2;
      if (!kUnrolled)
        for (int i = 0; i < N; ++i) interact<double, kFewM, MODE>(point(lev[0], i), px, py, pz, acc, c375);
      else if (lev[0] == 1 && t == 1) unrolled(integral_constant<int, 1>{}, integral_constant<int, 1>{});
      else if (lev[0] == 1 && t == 0) unrolled(integral_constant<int, 0>{}, integral_constant<int, 1>{});
      else if (lev[0] == 2 && t == 1) unrolled(integral_constant<int, 1>{}, integral_constant<int, 2>{});
      else if (lev[0] == 2 && t == 0) unrolled(integral_constant<int, 0>{}, integral_constant<int, 2>{});
      else
        for (int i = 0; i < N; ++i) interact<double, kFewM, MODE>(point(lev[0], i), px, py, pz, acc, c375);
      n_inter += (unsigned long long)N * mj;
      continue;
    }
#pragma unroll
    for (int j = 0; j < kFewM; ++j) {
      if (j >= mj) continue;
      if (lev[j] == 5) {
        Vec3 V[4];
        const int nv = load_polygon(p.type, p.verts, e, V);
        const double sg = __ldg(p.sigma + e);
        double ip;
        Vec3 ie;
        if constexpr (MODE == kModePhi) {
          analytic_integrals<false>(V, nv, Vec3{px[j], py[j], pz[j]}, ip, ie);
          acc.phi[j] += sg * ip;
        } else {
          analytic_integrals<true>(V, nv, Vec3{px[j], py[j], pz[j]}, ip, ie);
          acc.phi[j] += sg * ip;
          acc.ex[j] += sg * ie.x;
          acc.ey[j] += sg * ie.y;
          acc.ez[j] += sg * ie.z;
        }
        n_ana += 1;
      } else {
        const int N = rule_npts(t, lev[j]);
        for (int i = 0; i < N; ++i) {
          const double4 s = point(lev[j], i);
          if constexpr (MODE == kModePhi) interact_one_phi(s.x, s.y, s.z, s.w, px[j], py[j], pz[j], acc.phi[j], c375);
          else interact_one(s.x, s.y, s.z, s.w, px[j], py[j], pz[j], acc.phi[j], acc.ex[j], acc.ey[j], acc.ez[j], c375);
        }
        n_inter += N;
      }
    }
  }

  // lanes -> warp (shuffles) -> CTA (shared memory, fixed order) -> partial[blockIdx.x] -> the pass's last
  // CTA adds the CTAs' sums (fixed order too: a call is reproducible bit for bit) and writes the result
  __shared__ bool is_last;
#pragma unroll
  for (int j = 0; j < kFewM; ++j) {
    const double a = warp_sum_f64(acc.phi[j]);
    double bx = 0.0, by = 0.0, bz = 0.0;
    if constexpr (MODE != kModePhi) {
      bx = warp_sum_f64(acc.ex[j]);
      by = warp_sum_f64(acc.ey[j]);
      bz = warp_sum_f64(acc.ez[j]);
    }
    if (lane == 0) {
      red[warp][j][0] = a; red[warp][j][1] = bx; red[warp][j][2] = by; red[warp][j][3] = bz;
    }
  }
  __syncthreads();
  if (threadIdx.x < mj) {
    double4 s = make_double4(0, 0, 0, 0);
    for (int w = 0; w < kFewWarps; ++w) {
      s.x += red[w][threadIdx.x][0]; s.y += red[w][threadIdx.x][1];
      s.z += red[w][threadIdx.x][2]; s.w += red[w][threadIdx.x][3];
    }
    p.partial[(int64_t)blockIdx.x * p.m + j0 + threadIdx.x] = s;
  }
  if (p.counters) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      n_inter += __shfl_xor_sync(kFullMask, n_inter, o);
      n_ana += __shfl_xor_sync(kFullMask, n_ana, o);
    }
    if (lane == 0) {
      if (n_inter) atomicAdd(p.counters, n_inter);
      if (n_ana) atomicAdd(p.counters + 1, n_ana);
    }
  }
  __threadfence();  // this CTA's partial sums are visible before it counts itself done
  __syncthreads();
  if (threadIdx.x == 0) is_last = atomicAdd(p.done + blockIdx.y, 1u) == gridDim.x - 1;
  __syncthreads();
  if (!is_last) return;
  __threadfence();
  for (int j = 0; j < mj; ++j) {
    double4 s = make_double4(0, 0, 0, 0);
    for (int bx = threadIdx.x; bx < (int)gridDim.x; bx += blockDim.x) {
      const double2* v2 = reinterpret_cast<const double2*>(p.partial + (int64_t)bx * p.m + j0 + j);
      const double2 lo = __ldcg(v2), hi = __ldcg(v2 + 1);  // L2: written by other CTAs of this launch
      s.x += lo.x; s.y += lo.y; s.z += hi.x; s.w += hi.y;
    }
    s.x = warp_sum_f64(s.x); s.y = warp_sum_f64(s.y); s.z = warp_sum_f64(s.z); s.w = warp_sum_f64(s.w);
    __syncthreads();  // red[] of the previous point (or of the CTA's own sums) has been read
    if (lane == 0) {
      red[warp][0][0] = s.x; red[warp][0][1] = s.y; red[warp][0][2] = s.z; red[warp][0][3] = s.w;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
      double4 tsum = make_double4(0, 0, 0, 0);
      for (int w = 0; w < kFewWarps; ++w) {
        tsum.x += red[w][0][0]; tsum.y += red[w][0][1]; tsum.z += red[w][0][2]; tsum.w += red[w][0][3];
      }
      p.out_phi[j0 + j] = p.k * tsum.x;
      if (p.out_E) {
        p.out_E[3 * (j0 + j)] = p.k * tsum.y;
        p.out_E[3 * (j0 + j) + 1] = p.k * tsum.z;
        p.out_E[3 * (j0 + j) + 2] = p.k * tsum.w;
      }
    }
  }
}

// ------------------------------------------------------------------------------------------------
// Measurement helper (bemcub_inner_loop_rate): the very same consume() loop as the kernels above,
// fed from a window that is filled once - no TMA, no classification, no work queue.  Its rate is
// the ceiling the instruction mix of Eq. 4.1 allows on this GPU (register-file bandwidth and
// dependent-issue latency included), reported next to the DFMA-only peak.
template <int R>
__global__ void __launch_bounds__(kThreads, 1) inner_loop_kernel(const double4* __restrict__ pts, const double* __restrict__ field,
                                                                 int cnt, int trips, double4* __restrict__ out) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  double4* win = reinterpret_cast<double4*>(smem_raw) + (size_t)warp * kStages * kBuf;
  for (int i = lane; i < kStages * kBuf; i += 32) win[i] = pts[i];
  __syncwarp();
  const int64_t tile = (int64_t)blockIdx.x * kWarpsPerCta + warp;
  double px[R], py[R], pz[R];
  load_field_points<double, R>(field, (int64_t)gridDim.x * kWarpsPerCta * 32 * R, tile, lane, px, py, pz);
  Accum<double, R> tot;
  tot.zero();
  for (int t = 0; t < trips; ++t) {
    consume_into<R, kModePhiE>(win + (t & 1) * kBuf, cnt, px, py, pz, tot);
    __syncwarp();
  }
  store_partial<R, kModePhiE>(out, nullptr, (int64_t)gridDim.x * kWarpsPerCta * 32 * R, tile, lane, tot);
}

}  // namespace bemcub
