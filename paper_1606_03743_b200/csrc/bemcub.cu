// Host side of the bemcub C ABI (include/bemcub.h): context, scratch management, launch
// configuration.  All arithmetic of the hot path lives in the kernels included below; this file
// only validates arguments, sizes grids and enqueues kernels on the ctx stream.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>

#include <cuda_runtime.h>

#include "../../include/bemcub.h"
#include "kernels_assemble.cuh"
#include "kernels_eval.cuh"
#include "kernels_pairs.cuh"
#include "kernels_pre.cuh"
#include "kernels_paired.cuh"
#include "kernels_solve.cuh"
#include "kernels_sort.cuh"
#include "rules.h"

using namespace bemcub;

namespace {

// CODATA-2018 vacuum permittivity; the paper prints no value (reading 10).
const double kEps0 = 8.8541878128e-12;
const double kPi = 3.14159265358979323846;
inline double coulomb_k() { return 1.0 / (4.0 * kPi * kEps0); }

struct DevBuf {
  void* ptr = nullptr;
  size_t bytes = 0;
};

}  // namespace

constexpr int kCounterSlots = 8 + (kFewMaxM * 4 + 7) / 8;  // tallies, work queue, clock | eval_few_kernel's done counters
struct bemcub_ctx {
  int device = 0;
  cudaStream_t stream = nullptr;
  int num_sms = 148;
  // mesh
  int64_t n = 0;
  bool has_mesh = false;
  bool has_tri = false, has_rect = false;
  int64_t n_tri = 0, n_rect = 0;
  DevBuf type, verts, cenL, area;
  GeomStatus* d_status = nullptr;
  // expanded points per level (FP64 / FP32) and the stride they were built with
  DevBuf pts64[5], pts32[5];
  int stride[5] = {4, 7, 12, 19, 33};
  // rectangles in paired form per level (kernels_paired.cuh), with the sigma of the last call like pts64
  DevBuf pair64[5];
  bool charged_pair[5] = {false, false, false, false, false};
  int pair_np[5] = {0, 0, 0, 0, 0};  // pairs of the rectangle rule of each level (0: not pairable)
  DevBuf tri7;             // triangles' blocks for the 7-point rule in median form
  bool charged_tri7 = false, tri7_ok = false;
  int last_path = BEMCUB_PATH_NONE;
  int last_ipi = 0;  // FP64 instructions per interaction of the last call's kernels (0: FP32)
  // scratch
  DevBuf partial, partial_g;
  // charges of the last call that passed a sigma: which expanded levels still hold them, and the
  // sigma itself (the analytic branch needs it) - reused by calls with sigma == NULL
  bool charged64[5] = {false, false, false, false, false}, charged32[5] = {false, false, false, false, false};
  DevBuf sigma_keep;
  bool sigma_kept = false;
  DevBuf sort_key[2], sort_idx[2], sort_hist, sort_pts, sort_box;  // a2: Morton order of the field points
  const uint32_t* sort_perm = nullptr;  // result of the last sort, reusable by the solver for the same points
  const double* sort_src = nullptr;
  int64_t sort_m = 0;
  DevBuf solve_buf[6];  // GMRES: centroids, diagonal, basis, w, z/residual, small coefficient block
  // matrix fill: the rows of the last call in Morton order of their centroids (kept until the mesh changes)
  DevBuf asm_cen, asm_perm;
  int64_t asm_perm_row0 = -1, asm_perm_nrows = -1;
  DevBuf solve_matrix;   // the collocation matrix of a solve that keeps it (bemcub_solve_storage)
  int64_t solve_matrix_limit = 0;  // bytes; 0 = every solve is matrix-free
  DevBuf host_stage[5];  // device copies of host inputs/outputs for the *_host entry points
  unsigned long long* d_counters = nullptr;
  bemcub_stats stats{};
  bool counters_pending = false;
  bool counters_counted = true;  // false: the interaction count is known on the host (fixed rule); only the clock is read back
  // optional per-call timing of the dominant kernel (bemcub_set_timing)
  bool timing = false;
  bool timing_valid = false;
  cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};
};

namespace {

#define CUDA_TRY(expr)                         \
  do {                                         \
    cudaError_t _e = (expr);                   \
    if (_e != cudaSuccess) {                   \
      cudaGetLastError();                      \
      return _e == cudaErrorMemoryAllocation ? BEMCUB_ERR_NOMEM : BEMCUB_ERR_CUDA; \
    }                                          \
  } while (0)

int ensure(DevBuf& b, size_t bytes) {
  if (bytes <= b.bytes) return BEMCUB_OK;
  if (b.ptr) {
    cudaFree(b.ptr);
    b.ptr = nullptr;
    b.bytes = 0;
  }
  // grow with some headroom so that repeated slightly larger calls do not reallocate each time
  size_t want = bytes + bytes / 8 + 256;
  cudaError_t e = cudaMalloc(&b.ptr, want);
  if (e != cudaSuccess) {
    cudaGetLastError();
    want = bytes;
    e = cudaMalloc(&b.ptr, want);
  }
  if (e != cudaSuccess) {
    cudaGetLastError();
    b.ptr = nullptr;
    return BEMCUB_ERR_NOMEM;
  }
  b.bytes = want;
  return BEMCUB_OK;
}

void release(DevBuf& b) {
  if (b.ptr) cudaFree(b.ptr);
  b.ptr = nullptr;
  b.bytes = 0;
}

struct DeviceGuard {
  int prev = -1;
  bool ok = true;
  explicit DeviceGuard(int dev) {
    if (cudaGetDevice(&prev) != cudaSuccess) prev = -1;
    if (prev != dev) ok = (cudaSetDevice(dev) == cudaSuccess);
  }
  ~DeviceGuard() {
    int cur = -1;
    if (prev >= 0 && cudaGetDevice(&cur) == cudaSuccess && cur != prev) cudaSetDevice(prev);
  }
};

inline int rule_n(int type, int level) { return type == 0 ? bemcub_rules::kTriN[level] : bemcub_rules::kRectN[level]; }

void count_launch(bemcub_ctx* c, int k = 1) {
  c->stats.kernel_launches += k;
  c->stats.last_eval_launches += k;
}

int upload_tables() {
  double tri[75 * 4], rect[73 * 4];
  int toff[6], roff[6];
  int nt = 0, nr = 0;
  for (int l = 0; l < 5; ++l) {
    bemcub_rules::TriPoint tp[bemcub_rules::kMaxN];
    bemcub_rules::RectPoint rp[bemcub_rules::kMaxN];
    toff[l] = nt;
    roff[l] = nr;
    const int a = bemcub_rules::tri_points(l, tp), b = bemcub_rules::rect_points(l, rp);
    if (a != bemcub_rules::kTriN[l] || b != bemcub_rules::kRectN[l]) return BEMCUB_ERR_BAD_RULE;
    for (int i = 0; i < a; ++i, ++nt) {
      tri[4 * nt] = tp[i].la; tri[4 * nt + 1] = tp[i].lb; tri[4 * nt + 2] = tp[i].lc; tri[4 * nt + 3] = tp[i].w;
    }
    for (int i = 0; i < b; ++i, ++nr) {
      rect[4 * nr] = rp[i].x; rect[4 * nr + 1] = rp[i].y; rect[4 * nr + 2] = rp[i].w; rect[4 * nr + 3] = 0.0;
    }
  }
  toff[5] = nt;
  roff[5] = nr;
  for (int l = 0; l < 6; ++l)  // the unrolled point generator (rule_point_ct) has these offsets compiled in
    if (toff[l] != kTriOffCt[l] || roff[l] != kRectOffCt[l]) return BEMCUB_ERR_BAD_RULE;
  CUDA_TRY(cudaMemcpyToSymbol(c_tri_tab, tri, sizeof(tri)));
  CUDA_TRY(cudaMemcpyToSymbol(c_rect_tab, rect, sizeof(rect)));
  CUDA_TRY(cudaMemcpyToSymbol(c_tri_off, toff, sizeof(toff)));
  CUDA_TRY(cudaMemcpyToSymbol(c_rect_off, roff, sizeof(roff)));
  return BEMCUB_OK;
}

// Pairs (x, y), (-x, -y) of equal weight in the rectangle rules (kernels_paired.cuh): found in the tables
// themselves, so a rule that were not symmetric would simply not be paired (np = 0).
int upload_pair_tables(int np_out[5]) {
  double tab[5 * 16 * 4] = {0.0}, cw[5] = {0.0};
  int np[5] = {0, 0, 0, 0, 0};
  for (int l = 0; l < 5; ++l) {
    bemcub_rules::RectPoint rp[bemcub_rules::kMaxN];
    const int n = bemcub_rules::rect_points(l, rp);
    bool used[bemcub_rules::kMaxN] = {false};
    int k = 0;
    bool ok = true;
    for (int i = 0; i < n && ok; ++i) {
      if (used[i]) continue;
      used[i] = true;
      if (rp[i].x == 0.0 && rp[i].y == 0.0) {
        cw[l] += rp[i].w;
        continue;
      }
      int partner = -1;
      for (int j = i + 1; j < n; ++j)
        if (!used[j] && rp[j].x == -rp[i].x && rp[j].y == -rp[i].y && rp[j].w == rp[i].w) {
          partner = j;
          break;
        }
      if (partner < 0 || k >= 16) {
        ok = false;
        break;
      }
      used[partner] = true;
      tab[4 * (16 * l + k)] = rp[i].x;
      tab[4 * (16 * l + k) + 1] = rp[i].y;
      tab[4 * (16 * l + k) + 2] = rp[i].w;
      ++k;
    }
    np[l] = ok ? k : 0;
    if (!ok) cw[l] = 0.0;
    // eval_paired_kernel's consume_stage is instantiated per level for exactly these pair counts, with / without
    // a centre point (kernels_paired.cuh); a table that pairs differently is left to the plain point records
    static const int kPairsOfLevel[5] = {2, 3, 6, 8, 16};
    static const bool kCentreOfLevel[5] = {false, true, false, true, true};
    if (np[l] != 0 && (np[l] != kPairsOfLevel[l] || (cw[l] != 0.0) != kCentreOfLevel[l])) {
      np[l] = 0;
      cw[l] = 0.0;
      for (int k2 = 0; k2 < 16 * 4; ++k2) tab[4 * 16 * l + k2] = 0.0;
    }
  }
  CUDA_TRY(cudaMemcpyToSymbol(c_pair_tab, tab, sizeof(tab)));
  CUDA_TRY(cudaMemcpyToSymbol(c_pair_center_w, cw, sizeof(cw)));
  CUDA_TRY(cudaMemcpyToSymbol(c_pair_np, np, sizeof(np)));
  for (int l = 0; l < 5; ++l) np_out[l] = np[l];
  return BEMCUB_OK;
}

// The 7-point triangle rule as centroid + two orbits on the medians (kernels_paired.cuh): read off the table;
// *ok_out = false (and zeros uploaded) if the table does not have that structure.
int upload_tri7_tables(bool* ok_out) {
  bemcub_rules::TriPoint tp[bemcub_rules::kMaxN];
  const int n = bemcub_rules::tri_points(1, tp);
  double kappa[2] = {0.0, 0.0}, w[3] = {0.0, 0.0, 0.0};
  int seen[2][3] = {{0, 0, 0}, {0, 0, 0}};
  int norb = 0, ncen = 0;
  bool ok = n == 7;
  for (int i = 0; i < n && ok; ++i) {
    const double la = tp[i].la, lb = tp[i].lb, lc = tp[i].lc;
    if (la == lb && lb == lc) {
      w[0] = tp[i].w;
      ++ncen;
      continue;
    }
    int vtx;
    double a, b;
    if (lb == lc) { vtx = 0; a = la; b = lb; }
    else if (la == lc) { vtx = 1; a = lb; b = la; }
    else if (la == lb) { vtx = 2; a = lc; b = la; }
    else { ok = false; break; }
    const double k = a - b;
    int o = -1;
    for (int j = 0; j < norb; ++j)
      if (std::fabs(kappa[j] - k) <= 1e-14) o = j;
    if (o < 0) {
      if (norb == 2) { ok = false; break; }
      o = norb++;
      kappa[o] = k;
      w[1 + o] = tp[i].w;
    }
    if (tp[i].w != w[1 + o] || seen[o][vtx]) { ok = false; break; }
    seen[o][vtx] = 1;
  }
  ok = ok && ncen == 1 && norb == 2;
  for (int o = 0; o < 2 && ok; ++o) ok = seen[o][0] && seen[o][1] && seen[o][2];
  if (!ok) kappa[0] = kappa[1] = w[0] = w[1] = w[2] = 0.0;
  CUDA_TRY(cudaMemcpyToSymbol(c_tri7_kappa, kappa, sizeof(kappa)));
  CUDA_TRY(cudaMemcpyToSymbol(c_tri7_w, w, sizeof(w)));
  *ok_out = ok;
  return BEMCUB_OK;
}

// use_levels_mask -> level actually used for each wanted level (bemcub.h: next more accurate
// enabled one, else the most accurate enabled one below).
int build_policy(const bemcub_policy* hp, PolicyDev* out) {
  if (!hp) return BEMCUB_ERR_INVALID_ARG;
  const int mask = hp->use_levels_mask & 63;
  if (mask == 0) return BEMCUB_ERR_INVALID_ARG;
  for (int t = 0; t < 2; ++t)
    for (int b = 0; b < 5; ++b) {
      const double v = hp->dr[t][b];
      if (!(v >= 0.0) || !std::isfinite(v)) return BEMCUB_ERR_INVALID_ARG;
      if (b > 0 && v < hp->dr[t][b - 1]) return BEMCUB_ERR_INVALID_ARG;  // limits must not decrease
      out->dr[t][b] = v;
    }
  for (int want = 0; want <= 5; ++want) {
    int use = -1;
    for (int lv = want; lv <= 5 && use < 0; ++lv)
      if (mask & (1 << lv)) use = lv;
    for (int lv = want - 1; lv >= 0 && use < 0; --lv)
      if (mask & (1 << lv)) use = lv;
    out->map[want] = use;
  }
  out->allow_upgrade = hp->allow_upgrade ? 1 : 0;
  return BEMCUB_OK;
}

// Expanded points of one level, FP64 or FP32, into ctx-owned memory.
template <typename T>
int expand_level(bemcub_ctx* c, int level, const double* sigma, DevBuf& dst, const double* sigma_v = nullptr, int stride = 0,
                 double scale = 1.0) {
  typedef typename Point4<T>::type P4;
  if (stride == 0) stride = c->stride[level];
  const int64_t total = c->n * stride;
  int rc = ensure(dst, (size_t)std::max<int64_t>(total, 1) * sizeof(P4));
  if (rc) return rc;
  if (total == 0) return BEMCUB_OK;
  const int threads = 256;
  const int64_t blocks = (total + threads - 1) / threads;
  expand_kernel<T><<<(unsigned)blocks, threads, 0, c->stream>>>(
      c->n, level, stride, (const uint8_t*)c->type.ptr, (const double*)c->verts.ptr,
      (const double4*)c->cenL.ptr, (const double*)c->area.ptr, sigma, sigma_v, scale, (P4*)dst.ptr);
  count_launch(c);
  CUDA_TRY(cudaGetLastError());
  return BEMCUB_OK;
}

struct SplitPlan {
  int R;
  int64_t ntiles;
  int nsplit;
  int64_t elems_per_split;
  int64_t nitems;
  int grid;
};

// Work decomposition of the persistent evaluation kernels: item = (tile of 32R field points) x
// (split of the elements), pulled from an atomic queue by num_sms x 12 warps.  R (field points per
// lane) is as large as the problem allows while still giving every warp several items; the splits
// (multiples of 32 elements, the adaptive kernel's batch) make the items small enough that the
// tail of the launch - at most one item per warp - stays around one percent.
SplitPlan plan_splits(const bemcub_ctx* c, int64_t m, int max_r, bool adaptive) {
  SplitPlan s;
  const int64_t warps = (int64_t)c->num_sms * kWarpsPerCta;
  // shortest split: 64 elements where the rule is chosen per batch of 32 (adaptive), 32 elements for a fixed rule.
  // Round 3, fixed rule with 32 instead of 64: config 2 (6144 squares x 1e4 points) gets R = 2 and 30144 items,
  // kernel 0.504 -> 0.495 ms (N = 7), 2.311 -> 2.265 ms (N = 33); config 1 (1280 x 1000) 1280 instead of 640 items for
  // 1776 warps, kernel 38.8 -> 24.5 us; 1.5e6 x 1e4 unchanged (116.2 ms).  Asking for 8 instead of 16 items per warp,
  // or one CTA per item for grids below the SM count, changed nothing measurable.
  const int64_t max_by_len = std::max<int64_t>(1, c->n / (adaptive ? 64 : 32));
  s.R = 1;
  // Largest R that still leaves enough items per warp.  A fixed rule only gains from a larger R
  // (more chains per lane), so it may use many splits; in adaptive mode a larger tile of FEW field
  // points is also a looser tile (more upgraded elements), so R grows only when tiles are plentiful
  // (measured on 1.5e6 elements x 1e4 points: fixed rule +4 % with R = 4, adaptive -5 %; round 2, forcing
  // R = 4: that shape -6 %, the mat-vec of the level-5 icosphere solve -6 %).
  // (a fixed rule on a mesh of at most 64 elements - config 5's single element x 1e6 points: the items are so short
  // that their fixed cost counts, not their balance, so 4 items per warp are enough for a larger R: kernel 35.1 -> 22.5 us
  // at N = 7, 61.4 -> 55.3 us at N = 33)
  const int64_t split_cap = adaptive ? 64 : 512, per_warp = adaptive ? 8 : (c->n <= 64 ? 4 : 16);
  for (int R = max_r; R > 1; R >>= 1) {
    const int64_t nt = (m + 32 * R - 1) / (32 * R);
    if (nt * std::min<int64_t>(max_by_len, split_cap) >= per_warp * warps) {
      s.R = R;
      break;
    }
  }
  s.ntiles = (m + 32 * s.R - 1) / (32 * s.R);
  const int64_t target = warps * 64;
  int64_t ns = (target + s.ntiles - 1) / s.ntiles;
  const int64_t max_by_mem = std::max<int64_t>(1, (int64_t)(1ull << 31) / std::max<int64_t>(32 * m, 1));
  ns = std::max<int64_t>(1, std::min<int64_t>(std::min<int64_t>(ns, max_by_len), std::min<int64_t>(max_by_mem, 512)));
  int64_t eps = (c->n + ns - 1) / ns;
  eps = (eps + 31) / 32 * 32;
  if (eps < 32) eps = 32;
  s.elems_per_split = eps;
  s.nsplit = (int)std::max<int64_t>(1, (c->n + eps - 1) / eps);
  s.nitems = s.ntiles * s.nsplit;
  s.grid = (int)std::min<int64_t>(c->num_sms, (s.nitems + kWarpsPerCta - 1) / kWarpsPerCta);
  return s;
}

// launch configuration of eval_paired_kernel (measured on config 4)
// (config 4 at full size, final loops: 5 field points per lane x 8 warps/SM 7187 ms, 6 x 8 7265, 3 x 12 7282, 4 x 8 7314; with fewer
// field points the tiles must stay small: 3 x 12, then 1 x 12)
constexpr int kPairedR = 5, kPairedWarps = 8, kPairedMidR = 3, kPairedMidWarps = 12;

template <typename T, int R, int MODE = kModePhiE>
int launch_fixed(bemcub_ctx* c, const FixedParams& fp, const SplitPlan& sp) {
  const size_t smem = eval_smem_bytes<T>();  // opted in once per device by configure_kernels()
  eval_fixed_kernel<T, R, MODE><<<sp.grid, kThreads, smem, c->stream>>>(fp);
  count_launch(c);
  CUDA_TRY(cudaGetLastError());
  return BEMCUB_OK;
}

template <typename T, int R, int MODE = kModePhiE>
int launch_adaptive(bemcub_ctx* c, const AdaptiveParams& ap, const SplitPlan& sp) {
  const size_t smem = eval_smem_bytes<T>();
  eval_adaptive_kernel<T, R, MODE><<<sp.grid, kThreads, smem, c->stream>>>(ap);
  count_launch(c);
  CUDA_TRY(cudaGetLastError());
  return BEMCUB_OK;
}

// Opt-in to more than 48 KB of dynamic shared memory for every kernel instantiation that needs it,
// once per ctx (the attribute is per device), so that the asynchronous calls launch and nothing else.
template <typename K>
int opt_in_smem(K kernel, size_t bytes) {
  CUDA_TRY(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
  return BEMCUB_OK;
}
template <typename T, int MODE>
int configure_fixed() {
  int rc;
  const size_t b = eval_smem_bytes<T>();
  if ((rc = opt_in_smem(eval_fixed_kernel<T, 1, MODE>, b)) || (rc = opt_in_smem(eval_fixed_kernel<T, 2, MODE>, b))) return rc;
  if constexpr (MODE != kModeGrad) rc = opt_in_smem(eval_fixed_kernel<T, 4, MODE>, b);
  return rc;
}
template <typename T, int MODE>
int configure_adaptive() {
  int rc;
  const size_t b = eval_smem_bytes<T>();
  if ((rc = opt_in_smem(eval_adaptive_kernel<T, 1, MODE>, b)) || (rc = opt_in_smem(eval_adaptive_kernel<T, 2, MODE>, b))) return rc;
  if constexpr (MODE != kModeGrad) rc = opt_in_smem(eval_adaptive_kernel<T, 4, MODE>, b);
  return rc;
}
int configure_kernels() {
  int rc;
  if ((rc = configure_fixed<double, kModePhiE>()) || (rc = configure_fixed<double, kModePhi>()) ||
      (rc = configure_fixed<double, kModeGrad>()) || (rc = configure_fixed<float, kModePhiE>()) ||
      (rc = configure_fixed<float, kModePhi>()) || (rc = configure_adaptive<double, kModePhiE>()) ||
      (rc = configure_adaptive<double, kModePhi>()) || (rc = configure_adaptive<double, kModeGrad>()) ||
      (rc = configure_adaptive<float, kModePhiE>()) || (rc = configure_adaptive<float, kModePhi>()) ||
      (rc = opt_in_smem(assemble_kernel, assemble_smem_bytes())) ||
      (rc = opt_in_smem(eval_paired_kernel<kPairedR, kPairedWarps>, paired_smem_bytes<kPairedWarps>())) ||
      (rc = opt_in_smem(eval_paired_kernel<kPairedMidR, kPairedMidWarps>, paired_smem_bytes<kPairedMidWarps>())) ||
      (rc = opt_in_smem(eval_paired_kernel<1, kPairedMidWarps>, paired_smem_bytes<kPairedMidWarps>())) ||
      (rc = opt_in_smem(eval_paired_kernel<kPairedR, kPairedWarps, kModePhi>, paired_smem_bytes<kPairedWarps>())) ||
      (rc = opt_in_smem(eval_paired_kernel<kPairedMidR, kPairedMidWarps, kModePhi>, paired_smem_bytes<kPairedMidWarps>())) ||
      (rc = opt_in_smem(eval_paired_kernel<1, kPairedMidWarps, kModePhi>, paired_smem_bytes<kPairedMidWarps>())) ||
      (rc = opt_in_smem(inner_loop_kernel<4>, eval_smem_bytes<double>())))
    return rc;
  return BEMCUB_OK;
}

// a2 (first half): Morton order of the field points.  On success *perm is the device array with
// perm[j] = caller index of the j-th point in evaluation order and *sorted the permuted points.
int sort_field_points(bemcub_ctx* c, int64_t m, const double* field, const uint32_t** perm, const double** sorted) {
  int rc;
  const int nblocks = (int)((m + kSortChunk - 1) / kSortChunk);
  const size_t hist_entries = (size_t)kRadix * nblocks;
  for (int i = 0; i < 2; ++i)
    if ((rc = ensure(c->sort_key[i], (size_t)m * 4)) || (rc = ensure(c->sort_idx[i], (size_t)m * 4))) return rc;
  if ((rc = ensure(c->sort_hist, hist_entries * 4)) || (rc = ensure(c->sort_pts, (size_t)m * 24)) ||
      (rc = ensure(c->sort_box, 6 * sizeof(unsigned long long))))
    return rc;
  unsigned long long* box = (unsigned long long*)c->sort_box.ptr;
  CUDA_TRY(cudaMemsetAsync(box, 0xff, 3 * sizeof(unsigned long long), c->stream));
  CUDA_TRY(cudaMemsetAsync(box + 3, 0x00, 3 * sizeof(unsigned long long), c->stream));
  const int threads = 256;
  const unsigned mblocks = (unsigned)((m + threads - 1) / threads);
  bbox_kernel<<<std::min<unsigned>(mblocks, (unsigned)c->num_sms * 8), threads, 0, c->stream>>>(m, field, box);
  uint32_t* key[2] = {(uint32_t*)c->sort_key[0].ptr, (uint32_t*)c->sort_key[1].ptr};
  uint32_t* idx[2] = {(uint32_t*)c->sort_idx[0].ptr, (uint32_t*)c->sort_idx[1].ptr};
  morton_key_kernel<<<mblocks, threads, 0, c->stream>>>(m, field, box, key[0], idx[0]);
  count_launch(c, 2);
  int cur = 0;
  for (int shift = 0; shift < 30; shift += kRadixBits) {
    uint32_t* hist = (uint32_t*)c->sort_hist.ptr;
    radix_hist_kernel<<<nblocks, 32, 0, c->stream>>>(m, key[cur], shift, nblocks, hist);
    radix_scan_kernel<<<1, 1024, 0, c->stream>>>((int64_t)hist_entries, hist);
    radix_scatter_kernel<<<nblocks, 32, 0, c->stream>>>(m, key[cur], idx[cur], shift, nblocks, hist, key[cur ^ 1],
                                                        idx[cur ^ 1]);
    count_launch(c, 3);
    cur ^= 1;
  }
  gather_points_kernel<<<mblocks, threads, 0, c->stream>>>(m, field, idx[cur], (double*)c->sort_pts.ptr);
  count_launch(c);
  CUDA_TRY(cudaGetLastError());
  *perm = idx[cur];
  *sorted = (const double*)c->sort_pts.ptr;
  return BEMCUB_OK;
}

// ev[0] call start, ev[1] before the dominant kernel, ev[2] after it, ev[3] call end
void mark(bemcub_ctx* c, int i) {
  if (c->timing) cudaEventRecord(c->ev[i], c->stream);
}

void refresh_counters(bemcub_ctx* c) {
  if (!c->counters_pending) return;
  unsigned long long h[6] = {0, 0, 0, 0, 0, 0};
  cudaStreamSynchronize(c->stream);
  if (cudaMemcpy(h, c->d_counters, sizeof(h), cudaMemcpyDeviceToHost) == cudaSuccess) {
    if (c->counters_counted) {
      c->stats.point_interactions = (int64_t)h[0];
      c->stats.analytic_pairs = (int64_t)h[1];
    }
    c->stats.kernel_cycles = (int64_t)h[4];
    c->stats.kernel_ns = (int64_t)h[5];
    c->stats.fp64_instructions = c->stats.point_interactions * c->last_ipi - (int64_t)h[3];  // h[3]: saved by the paired form
  }
  c->counters_pending = false;
}

}  // namespace

extern "C" {

const char* bemcub_strerror(int code) {
  switch (code) {
    case BEMCUB_OK: return "ok";
    case BEMCUB_ERR_INVALID_ARG: return "invalid argument";
    case BEMCUB_ERR_DEGENERATE_ELEMENT: return "degenerate element (zero area or zero side)";
    case BEMCUB_ERR_NOT_RECTANGLE: return "rectangle sides are not orthogonal";
    case BEMCUB_ERR_BAD_RULE: return "unknown rule id / element type";
    case BEMCUB_ERR_CUDA: return "CUDA error";
    case BEMCUB_ERR_NOMEM: return "out of device memory";
    case BEMCUB_ERR_NO_ELEMENTS: return "no mesh: call bemcub_set_elements first";
    case BEMCUB_ERR_NOT_CONVERGED: return "iteration stopped at the mat-vec limit before reaching the tolerance";
    case BEMCUB_ERR_TOO_MANY_ELEMENTS:
      return "matrix fill: the mesh has more than 2^25 = 33,554,432 elements (columns), even for a window of a few rows";
    case BEMCUB_ERR_FIXED_SCRATCH:
      return "bemcub_eval_few_noalloc: beyond its fixed scratch (at most 64 field points per call, devices of at most 160 SMs)";
  }
  return "unknown error code";
}

int bemcub_rule_info(int elem_type, int rule_id, int* npts, int* degree) {
  if ((elem_type != BEMCUB_TRI && elem_type != BEMCUB_RECT) || rule_id < 0 || rule_id > 4) return BEMCUB_ERR_BAD_RULE;
  if (npts) *npts = rule_n(elem_type, rule_id);
  if (degree) *degree = elem_type == 0 ? bemcub_rules::kTriDegree[rule_id] : bemcub_rules::kRectDegree[rule_id];
  return BEMCUB_OK;
}

int bemcub_rule_points(int elem_type, int rule_id, double* host_coords, double* host_w) {
  if ((elem_type != BEMCUB_TRI && elem_type != BEMCUB_RECT) || rule_id < 0 || rule_id > 4) return BEMCUB_ERR_BAD_RULE;
  if (!host_coords || !host_w) return BEMCUB_ERR_INVALID_ARG;
  if (elem_type == BEMCUB_TRI) {
    bemcub_rules::TriPoint tp[bemcub_rules::kMaxN];
    const int n = bemcub_rules::tri_points(rule_id, tp);
    for (int i = 0; i < n; ++i) {
      host_coords[3 * i] = tp[i].la; host_coords[3 * i + 1] = tp[i].lb; host_coords[3 * i + 2] = tp[i].lc;
      host_w[i] = tp[i].w;
    }
  } else {
    bemcub_rules::RectPoint rp[bemcub_rules::kMaxN];
    const int n = bemcub_rules::rect_points(rule_id, rp);
    for (int i = 0; i < n; ++i) {
      host_coords[2 * i] = rp[i].x; host_coords[2 * i + 1] = rp[i].y;
      host_w[i] = rp[i].w;
    }
  }
  return BEMCUB_OK;
}

int bemcub_default_policy(bemcub_policy* hp, int want_field) {
  if (!hp) return BEMCUB_ERR_INVALID_ARG;
  // L159: printed triangle-potential limits; Phi+E limits per DESIGN.md reading 7
  static const double pot[5] = {3, 8, 20, 80, 1500};
  static const double ftri[5] = {4, 10, 25, 100, 2000};
  static const double frect[5] = {6, 15, 40, 150, 3000};
  // BEMCUB_POLICY_FIELD_F32: where each rule's own error of the field falls below the FP32 rounding
  // floor (1e-7; profiles/r2_accuracy_sweep.txt) - N = 33 is never worth its points in FP32 on triangles
  static const double f32tri[5] = {2, 2, 3, 6, 25};
  static const double f32rect[5] = {2, 3, 4, 8, 30};
  if (want_field < 0 || want_field > BEMCUB_POLICY_FIELD_F32) return BEMCUB_ERR_INVALID_ARG;
  for (int b = 0; b < 5; ++b) {
    hp->dr[0][b] = want_field == BEMCUB_POLICY_FIELD_F32 ? f32tri[b] : want_field ? ftri[b] : pot[b];
    hp->dr[1][b] = want_field == BEMCUB_POLICY_FIELD_F32 ? f32rect[b] : want_field ? frect[b] : pot[b];
  }
  hp->allow_upgrade = 1;
  hp->use_levels_mask = 63;
  return BEMCUB_OK;
}

int bemcub_create(bemcub_ctx** out_ctx, int device, void* cuda_stream) {
  if (!out_ctx) return BEMCUB_ERR_INVALID_ARG;
  *out_ctx = nullptr;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) {
    cudaGetLastError();
    return BEMCUB_ERR_CUDA;  // no CPU fallback: the library is useless without a GPU
  }
  DeviceGuard g(device);
  if (!g.ok) return BEMCUB_ERR_CUDA;
  bemcub_ctx* c = new (std::nothrow) bemcub_ctx();
  if (!c) return BEMCUB_ERR_NOMEM;
  c->device = device;
  c->stream = (cudaStream_t)cuda_stream;
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) {
    delete c;
    return BEMCUB_ERR_CUDA;
  }
  c->num_sms = prop.multiProcessorCount;
  int rc = upload_tables();
  if (rc == BEMCUB_OK) rc = upload_pair_tables(c->pair_np);
  if (rc == BEMCUB_OK) rc = upload_tri7_tables(&c->tri7_ok);
  if (rc == BEMCUB_OK) rc = configure_kernels();
  if (rc == BEMCUB_OK && cudaMalloc(&c->d_status, sizeof(GeomStatus)) != cudaSuccess) rc = BEMCUB_ERR_NOMEM;
  if (rc == BEMCUB_OK && cudaMalloc(&c->d_counters, kCounterSlots * sizeof(unsigned long long)) != cudaSuccess) rc = BEMCUB_ERR_NOMEM;
  if (rc != BEMCUB_OK) {
    bemcub_destroy(c);
    return rc;
  }
  *out_ctx = c;
  return BEMCUB_OK;
}

int bemcub_destroy(bemcub_ctx* c) {
  if (!c) return BEMCUB_OK;
  DeviceGuard g(c->device);
  cudaStreamSynchronize(c->stream);
  release(c->type); release(c->verts); release(c->cenL); release(c->area); release(c->partial); release(c->partial_g); release(c->sigma_keep);
  for (int l = 0; l < 5; ++l) { release(c->pts64[l]); release(c->pts32[l]); release(c->host_stage[l]); release(c->pair64[l]); }
  release(c->tri7);
  for (int i = 0; i < 2; ++i) { release(c->sort_key[i]); release(c->sort_idx[i]); }
  release(c->sort_hist); release(c->sort_pts); release(c->sort_box);
  for (int i = 0; i < 6; ++i) release(c->solve_buf[i]);
  release(c->solve_matrix);
  release(c->asm_cen); release(c->asm_perm);
  if (c->d_status) cudaFree(c->d_status);
  if (c->d_counters) cudaFree(c->d_counters);
  for (int i = 0; i < 4; ++i)
    if (c->ev[i]) cudaEventDestroy(c->ev[i]);
  delete c;
  return BEMCUB_OK;
}

int bemcub_set_elements(bemcub_ctx* c, int64_t n, const uint8_t* type, const double* verts) {
  if (!c || n < 0 || (n > 0 && (!type || !verts))) return BEMCUB_ERR_INVALID_ARG;
  DeviceGuard g(c->device);
  c->has_mesh = false;
  c->n = 0;
  c->sort_perm = nullptr;
  c->asm_perm_row0 = c->asm_perm_nrows = -1;
  c->sigma_kept = false;
  for (int l = 0; l < 5; ++l) c->charged64[l] = c->charged32[l] = c->charged_pair[l] = false;
  c->charged_tri7 = false;
  int rc;
  const size_t nn = (size_t)std::max<int64_t>(n, 1);
  if ((rc = ensure(c->type, nn)) || (rc = ensure(c->verts, nn * 72)) || (rc = ensure(c->cenL, nn * sizeof(double4))) ||
      (rc = ensure(c->area, nn * 8)))
    return rc;
  GeomStatus st = {0, 0, 0, 0};
  if (n > 0) {
    CUDA_TRY(cudaMemcpyAsync(c->type.ptr, type, (size_t)n, cudaMemcpyDeviceToDevice, c->stream));
    CUDA_TRY(cudaMemcpyAsync(c->verts.ptr, verts, (size_t)n * 72, cudaMemcpyDeviceToDevice, c->stream));
    CUDA_TRY(cudaMemsetAsync(c->d_status, 0, sizeof(GeomStatus), c->stream));
    const int threads = 256;
    geometry_kernel<<<(unsigned)((n + threads - 1) / threads), threads, 0, c->stream>>>(
        n, (const uint8_t*)c->type.ptr, (const double*)c->verts.ptr, (double4*)c->cenL.ptr, (double*)c->area.ptr,
        c->d_status);
    c->stats.kernel_launches += 1;
    CUDA_TRY(cudaGetLastError());
    CUDA_TRY(cudaMemcpyAsync(&st, c->d_status, sizeof(st), cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(cudaStreamSynchronize(c->stream));
    if (st.code != 0) return st.code;  // -1 invalid type, -2 degenerate, -3 not a rectangle
  }
  c->n = n;
  c->n_tri = (int64_t)st.n_tri;
  c->n_rect = (int64_t)st.n_rect;
  c->has_tri = st.n_tri != 0;
  c->has_rect = st.n_rect != 0;
  for (int l = 0; l < 5; ++l)
    c->stride[l] = std::max(c->has_tri ? bemcub_rules::kTriN[l] : 0, c->has_rect ? bemcub_rules::kRectN[l] : 0);
  if (n == 0)
    for (int l = 0; l < 5; ++l) c->stride[l] = bemcub_rules::kTriN[l];
  c->has_mesh = true;
  return BEMCUB_OK;
}

int bemcub_get_geometry(bemcub_ctx* c, double* out_cen, double* out_area, double* out_L) {
  if (!c) return BEMCUB_ERR_INVALID_ARG;
  if (!c->has_mesh) return BEMCUB_ERR_NO_ELEMENTS;
  DeviceGuard g(c->device);
  if (c->n == 0) return BEMCUB_OK;
  if (out_cen)
    CUDA_TRY(cudaMemcpy2DAsync(out_cen, 24, c->cenL.ptr, 32, 24, (size_t)c->n, cudaMemcpyDeviceToDevice, c->stream));
  if (out_L)
    CUDA_TRY(cudaMemcpy2DAsync(out_L, 8, (const char*)c->cenL.ptr + 24, 32, 8, (size_t)c->n, cudaMemcpyDeviceToDevice,
                               c->stream));
  if (out_area) CUDA_TRY(cudaMemcpyAsync(out_area, c->area.ptr, (size_t)c->n * 8, cudaMemcpyDeviceToDevice, c->stream));
  return BEMCUB_OK;
}

int bemcub_expand_points(bemcub_ctx* c, const double* sigma, int rule_id, double* out_xyzq, int* out_stride) {
  if (!c || !out_xyzq) return BEMCUB_ERR_INVALID_ARG;
  if (!c->has_mesh) return BEMCUB_ERR_NO_ELEMENTS;
  if (rule_id < 0 || rule_id > 4) return BEMCUB_ERR_BAD_RULE;
  DeviceGuard g(c->device);
  if (out_stride) *out_stride = c->stride[rule_id];
  c->charged64[rule_id] = false;
  int rc = expand_level<double>(c, rule_id, sigma, c->pts64[rule_id]);
  if (rc) return rc;
  if (c->n > 0)
    CUDA_TRY(cudaMemcpyAsync(out_xyzq, c->pts64[rule_id].ptr, (size_t)c->n * c->stride[rule_id] * 32,
                             cudaMemcpyDeviceToDevice, c->stream));
  return BEMCUB_OK;
}

}  // extern "C"

namespace {

// bemcub_eval and bemcub_eval_gradient (out_G != nullptr) share everything but the accumulators.
int eval_common(bemcub_ctx* c, const double* sigma, int rule_id, const bemcub_policy* host_policy, int64_t m,
                const double* field_pts, double* out_phi, double* out_E, double* out_G, int precision,
                bool reuse_sort = false, const double* sigma_v = nullptr) {
  if (!c || m < 0) return BEMCUB_ERR_INVALID_ARG;
  if (!c->has_mesh) return BEMCUB_ERR_NO_ELEMENTS;
  if (rule_id < -1 || rule_id > 4) return BEMCUB_ERR_BAD_RULE;
  if (precision != BEMCUB_F64 && precision != BEMCUB_F32) return BEMCUB_ERR_INVALID_ARG;
  if (m == 0) return BEMCUB_OK;
  if (!field_pts || (!out_phi && !out_E && !out_G)) return BEMCUB_ERR_INVALID_ARG;
  const bool reuse = !sigma && !sigma_v;  // sigma == NULL: the charges of the previous call
  const bool adaptive = rule_id == BEMCUB_RULE_ADAPTIVE;
  const bool grad = out_G != nullptr;
  if (grad && precision != BEMCUB_F64) return BEMCUB_ERR_INVALID_ARG;  // the gradient is FP64 only
  PolicyDev pol;
  if (adaptive) {
    int rc = build_policy(host_policy, &pol);
    if (rc) return rc;
    // derivatives exist for the point charges only (L273): no analytic branch in a gradient call
    if ((grad || sigma_v) && (host_policy->use_levels_mask & (1 << BEMCUB_LEVEL_ANALYTIC))) return BEMCUB_ERR_INVALID_ARG;
  }
  DeviceGuard g(c->device);
  c->stats.last_eval_launches = 0;
  int rc;

  if (c->n == 0) {  // empty mesh: zero potential and field
    if (out_phi) CUDA_TRY(cudaMemsetAsync(out_phi, 0, (size_t)m * 8, c->stream));
    if (out_E) CUDA_TRY(cudaMemsetAsync(out_E, 0, (size_t)m * 24, c->stream));
    if (out_G) CUDA_TRY(cudaMemsetAsync(out_G, 0, (size_t)m * 48, c->stream));
    c->stats.point_interactions = 0;
    c->stats.analytic_pairs = 0;
    return BEMCUB_OK;
  }

  c->timing_valid = false;
  mark(c, 0);
  // a1: expand the levels this call needs, sigma folded in - or, with sigma == NULL, check that the
  // previous call left them there (tracking evaluates the same charges at point after point)
  bool need[5] = {false, false, false, false, false};
  if (adaptive) {
    for (int l = 0; l < 5; ++l)
      for (int w = 0; w <= 5; ++w) need[l] |= (pol.map[w] == l);
  } else {
    need[rule_id] = true;
  }
  // Few field points (tracking-style calls): elements across the lanes, per-pair rule choice,
  // warp-shuffle reduction (eval_few_kernel); no tiles, hence no sort.
  // What a ctx keeps between calls is the sigma of the last call that brought one (sigma_keep);
  // the expanded levels are a cache of it (charged[l] = level l holds exactly those charges).
  if (reuse) {
    if (!c->sigma_kept) return BEMCUB_ERR_INVALID_ARG;
    sigma = (const double*)c->sigma_keep.ptr;
  } else {
    for (int l = 0; l < 5; ++l) c->charged64[l] = c->charged32[l] = c->charged_pair[l] = false;  // other charges from now on
    c->charged_tri7 = false;
    c->sigma_kept = false;
    if (sigma) {
      if ((rc = ensure(c->sigma_keep, (size_t)c->n * 8))) return rc;
      CUDA_TRY(cudaMemcpyAsync(c->sigma_keep.ptr, sigma, (size_t)c->n * 8, cudaMemcpyDeviceToDevice, c->stream));
      c->sigma_kept = true;
    }
  }
  const bool few = !grad && precision == BEMCUB_F64 && m <= kFewMaxM;
  if (few) {
    // a pass takes 4 field points (2 or 1 if that is all there is: no work on clamped duplicates)
    const int per_pass = m >= 3 ? kFewM : (int)m;
    const int blocks = c->num_sms * 2;
    if ((rc = ensure(c->partial, (size_t)blocks * (size_t)m * sizeof(double4)))) return rc;
    FewParams fw;
    fw.cenL = (const double4*)c->cenL.ptr;
    fw.type = (const uint8_t*)c->type.ptr;
    fw.verts = (const double*)c->verts.ptr;
    fw.sigma = sigma;
    fw.n = c->n;
    if (adaptive) fw.pol = pol;
    fw.rule = adaptive ? -1 : rule_id;
    fw.field = field_pts;
    fw.m = m;
    fw.partial = (double4*)c->partial.ptr;
    fw.counters = c->d_counters;
    fw.area = (const double*)c->area.ptr;
    fw.sigma_v = sigma_v;
    fw.done = reinterpret_cast<unsigned*>(c->d_counters + 8);  // one per pass (<= kFewMaxM)
    fw.k = coulomb_k();
    fw.out_phi = out_phi;
    fw.out_E = out_E;
    CUDA_TRY(cudaMemsetAsync(c->d_counters, 0, kCounterSlots * sizeof(unsigned long long), c->stream));
    mark(c, 1);
    const dim3 grid((unsigned)blocks, (unsigned)((m + per_pass - 1) / per_pass));
    // points on the fly from the vertices (measured faster than reading kept points: 121 instead of
    // 260 bytes per element; 0.119 vs 0.144 ms for one field point on 1e6 elements)
    const int threads = kFewWarps * 32;
    if (out_E) {
      if (per_pass == 1) eval_few_kernel<kModePhiE, 1><<<grid, threads, 0, c->stream>>>(fw);
      else if (per_pass == 2) eval_few_kernel<kModePhiE, 2><<<grid, threads, 0, c->stream>>>(fw);
      else eval_few_kernel<kModePhiE, kFewM><<<grid, threads, 0, c->stream>>>(fw);
    } else {
      if (per_pass == 1) eval_few_kernel<kModePhi, 1><<<grid, threads, 0, c->stream>>>(fw);
      else if (per_pass == 2) eval_few_kernel<kModePhi, 2><<<grid, threads, 0, c->stream>>>(fw);
      else eval_few_kernel<kModePhi, kFewM><<<grid, threads, 0, c->stream>>>(fw);
    }
    count_launch(c);
    CUDA_TRY(cudaGetLastError());
    mark(c, 2);
    mark(c, 3);  // a6 (sum over the CTAs, k) happens in the last CTA of every pass
    c->last_path = BEMCUB_PATH_FEW;
    c->stats.field_points_per_lane = 0;
    c->last_ipi = out_E ? 18 : 12;
    c->timing_valid = c->timing;
    c->counters_pending = true;
    c->counters_counted = true;
    return BEMCUB_OK;
  }

  bool* charged = precision == BEMCUB_F64 ? c->charged64 : c->charged32;
  for (int l = 0; l < 5; ++l) {
    if (!need[l] || charged[l]) continue;
    if (precision == BEMCUB_F64) rc = expand_level<double>(c, l, sigma, c->pts64[l], sigma_v);
    else rc = expand_level<float>(c, l, sigma, c->pts32[l], sigma_v);
    if (rc) return rc;
    charged[l] = sigma_v == nullptr;  // a linear density is not kept (sigma_keep holds constants only)
  }

  // Rectangles in paired form (kernels_paired.cuh): FP64 Phi + E with the distance-ratio choice, a constant
  // density, a policy whose analytic branch covers the rectangles below a distance ratio of 2 at least (so
  // that |d| < |D| wherever a pair is evaluated), and field points enough for tiles of 32 kPairedR.
  bool paired = false, tri7 = false;
  if (adaptive && !grad && precision == BEMCUB_F64 && !sigma_v && pol.map[5] == 5) {
    if (c->has_rect && pol.dr[1][0] >= 2.0)
      for (int l = 0; l < 5; ++l) paired |= need[l] && c->pair_np[l] > 0;
    // ... and the 7-point triangle rule in median form, under the same condition on the triangles' analytic limit
    // (a potential-only call on a mesh of triangles alone is typically the mat-vec of a solve: field points on the mesh
    // itself, where the 7-point rule is never reached - the level-5 icosphere solve was 19 % slower through this kernel)
    tri7 = c->has_tri && c->tri7_ok && need[1] && pol.dr[0][0] >= 2.0 && (out_E || paired);
    paired |= tri7;
    // (with fewer field points: one per lane, as the plain kernel does - plan_splits gives 3 or 1)
  }
  if (paired && tri7 && !c->charged_tri7) {
    if ((rc = ensure(c->tri7, (size_t)c->n * kTri7Units * sizeof(double4)))) return rc;
    expand_tri7_kernel<<<(unsigned)((4 * c->n + 255) / 256), 256, 0, c->stream>>>(
        c->n, (const uint8_t*)c->type.ptr, (const double*)c->verts.ptr, (const double4*)c->cenL.ptr, (const double*)c->area.ptr,
        sigma, (double*)c->tri7.ptr);
    count_launch(c);
    CUDA_TRY(cudaGetLastError());
    c->charged_tri7 = true;
  }
  if (paired) {
    for (int l = 0; l < 5; ++l) {
      const int np = (c->has_rect && pol.dr[1][0] >= 2.0) ? c->pair_np[l] : 0;
      if (!need[l] || np == 0 || c->charged_pair[l]) continue;
      if ((rc = ensure(c->pair64[l], (size_t)c->n * pair_units(np) * sizeof(double4)))) return rc;
      const int64_t total = c->n * (np + 1);
      expand_pairs_kernel<<<(unsigned)((total + 255) / 256), 256, 0, c->stream>>>(
          c->n, l, np, (const uint8_t*)c->type.ptr, (const double*)c->verts.ptr, (const double4*)c->cenL.ptr,
          (const double*)c->area.ptr, sigma, (double*)c->pair64[l].ptr);
      count_launch(c);
      CUDA_TRY(cudaGetLastError());
      c->charged_pair[l] = true;
    }
  }
  SplitPlan sp = plan_splits(c, m, paired ? kPairedR : (grad ? 2 : 4), adaptive);  // R = 6 was measured: 2 % slower than R = 4 in the full kernel
  if (paired && sp.R != kPairedR) sp = plan_splits(c, m, kPairedMidR, adaptive);  // 5, else 3, else 1 field points per lane
  if ((rc = ensure(c->partial, (size_t)sp.nsplit * (size_t)m * sizeof(double4)))) return rc;
  if (grad && (rc = ensure(c->partial_g, (size_t)sp.nsplit * (size_t)m * 48))) return rc;
  // a2: tiles of spatially close field points (adaptive mode; a fixed rule has nothing to choose)
  const uint32_t* perm = nullptr;
  if (adaptive && m > 32 && m < ((int64_t)1 << 31)) {
    if (reuse_sort && c->sort_perm && c->sort_src == field_pts && c->sort_m == m) {
      perm = c->sort_perm;  // the solver evaluates at the same centroids every iteration
      field_pts = (const double*)c->sort_pts.ptr;
    } else {
      const double* src = field_pts;
      c->sort_perm = nullptr;
      if ((rc = sort_field_points(c, m, field_pts, &perm, &field_pts))) return rc;
      c->sort_perm = perm;
      c->sort_src = src;
      c->sort_m = m;
    }
  }
  mark(c, 1);

  if (!adaptive) {
    FixedParams fp;
    fp.pts = precision == BEMCUB_F64 ? c->pts64[rule_id].ptr : c->pts32[rule_id].ptr;
    fp.npts = c->n * c->stride[rule_id];
    fp.pts_per_split = sp.elems_per_split * c->stride[rule_id];
    fp.field = field_pts;
    fp.m = m;
    fp.partial = (double4*)c->partial.ptr;
    fp.partial_g = (double*)c->partial_g.ptr;
    fp.split_stride = m;
    fp.ntiles = sp.ntiles;
    fp.nitems = sp.nitems;
    fp.queue = c->d_counters + 2;
    fp.counters = c->d_counters;
    CUDA_TRY(cudaMemsetAsync(c->d_counters, 0, 8 * sizeof(unsigned long long), c->stream));
    const bool phi_only = !grad && !out_E;
    if (grad)
      rc = sp.R == 2 ? launch_fixed<double, 2, kModeGrad>(c, fp, sp) : launch_fixed<double, 1, kModeGrad>(c, fp, sp);
    else if (precision == BEMCUB_F64 && phi_only)
      rc = sp.R == 4 ? launch_fixed<double, 4, kModePhi>(c, fp, sp) : sp.R == 2 ? launch_fixed<double, 2, kModePhi>(c, fp, sp) : launch_fixed<double, 1, kModePhi>(c, fp, sp);
    else if (precision == BEMCUB_F64)
      rc = sp.R == 4 ? launch_fixed<double, 4>(c, fp, sp) : sp.R == 2 ? launch_fixed<double, 2>(c, fp, sp) : launch_fixed<double, 1>(c, fp, sp);
    else if (phi_only)
      rc = sp.R == 4 ? launch_fixed<float, 4, kModePhi>(c, fp, sp) : sp.R == 2 ? launch_fixed<float, 2, kModePhi>(c, fp, sp) : launch_fixed<float, 1, kModePhi>(c, fp, sp);
    else
      rc = sp.R == 4 ? launch_fixed<float, 4>(c, fp, sp) : sp.R == 2 ? launch_fixed<float, 2>(c, fp, sp) : launch_fixed<float, 1>(c, fp, sp);
    if (rc) return rc;
    // point-charge interactions of a fixed rule: every element's own N at every field point
    c->stats.point_interactions =
        (c->n_tri * bemcub_rules::kTriN[rule_id] + c->n_rect * bemcub_rules::kRectN[rule_id]) * m;
    c->stats.analytic_pairs = 0;
    c->counters_pending = true;
    c->counters_counted = false;
  } else {
    AdaptiveParams ap;
    for (int l = 0; l < 5; ++l) {
      ap.lvl_pts[l] = precision == BEMCUB_F64 ? c->pts64[l].ptr : c->pts32[l].ptr;
      ap.stride[l] = c->stride[l];
    }
    ap.cenL = (const double4*)c->cenL.ptr;
    ap.type = (const uint8_t*)c->type.ptr;
    ap.verts = (const double*)c->verts.ptr;
    ap.sigma = sigma;
    ap.n = c->n;
    ap.elems_per_split = sp.elems_per_split;
    ap.pol = pol;
    ap.field = field_pts;
    ap.m = m;
    ap.partial = (double4*)c->partial.ptr;
    ap.partial_g = (double*)c->partial_g.ptr;
    ap.split_stride = m;
    ap.ntiles = sp.ntiles;
    ap.nitems = sp.nitems;
    ap.queue = c->d_counters + 2;
    ap.counters = c->d_counters;
    CUDA_TRY(cudaMemsetAsync(c->d_counters, 0, 8 * sizeof(unsigned long long), c->stream));
    if (paired) {
      PairedParams pq;
      pq.ad = ap;
      for (int l = 0; l < 5; ++l) {
        pq.pair_np[l] = (need[l] && c->has_rect && pol.dr[1][0] >= 2.0) ? c->pair_np[l] : 0;
        pq.pair_pts[l] = (const double4*)c->pair64[l].ptr;
      }
      pq.tri7_pts = tri7 ? (const double4*)c->tri7.ptr : nullptr;
      const int wpc = sp.R == kPairedR ? kPairedWarps : kPairedMidWarps;
      const int grid = (int)std::min<int64_t>(c->num_sms, (sp.nitems + wpc - 1) / wpc);
      const size_t sm_big = paired_smem_bytes<kPairedWarps>(), sm_mid = paired_smem_bytes<kPairedMidWarps>();
      if (out_E) {
        if (sp.R == kPairedR) eval_paired_kernel<kPairedR, kPairedWarps><<<grid, kPairedWarps * 32, sm_big, c->stream>>>(pq);
        else if (sp.R == kPairedMidR) eval_paired_kernel<kPairedMidR, kPairedMidWarps><<<grid, kPairedMidWarps * 32, sm_mid, c->stream>>>(pq);
        else eval_paired_kernel<1, kPairedMidWarps><<<grid, kPairedMidWarps * 32, sm_mid, c->stream>>>(pq);
      } else {  // potential only (the mat-vec of bemcub_solve)
        if (sp.R == kPairedR) eval_paired_kernel<kPairedR, kPairedWarps, kModePhi><<<grid, kPairedWarps * 32, sm_big, c->stream>>>(pq);
        else if (sp.R == kPairedMidR)
          eval_paired_kernel<kPairedMidR, kPairedMidWarps, kModePhi><<<grid, kPairedMidWarps * 32, sm_mid, c->stream>>>(pq);
        else eval_paired_kernel<1, kPairedMidWarps, kModePhi><<<grid, kPairedMidWarps * 32, sm_mid, c->stream>>>(pq);
      }
      count_launch(c);
      CUDA_TRY(cudaGetLastError());
      rc = BEMCUB_OK;
    } else if (grad) rc = sp.R == 2 ? launch_adaptive<double, 2, kModeGrad>(c, ap, sp) : launch_adaptive<double, 1, kModeGrad>(c, ap, sp);
    else if (precision == BEMCUB_F64 && !out_E)
      rc = sp.R == 4 ? launch_adaptive<double, 4, kModePhi>(c, ap, sp) : sp.R == 2 ? launch_adaptive<double, 2, kModePhi>(c, ap, sp) : launch_adaptive<double, 1, kModePhi>(c, ap, sp);
    else if (precision == BEMCUB_F64)
      rc = sp.R == 4 ? launch_adaptive<double, 4>(c, ap, sp) : sp.R == 2 ? launch_adaptive<double, 2>(c, ap, sp) : launch_adaptive<double, 1>(c, ap, sp);
    else if (!out_E)
      rc = sp.R == 4 ? launch_adaptive<float, 4, kModePhi>(c, ap, sp) : sp.R == 2 ? launch_adaptive<float, 2, kModePhi>(c, ap, sp) : launch_adaptive<float, 1, kModePhi>(c, ap, sp);
    else
      rc = sp.R == 4 ? launch_adaptive<float, 4>(c, ap, sp) : sp.R == 2 ? launch_adaptive<float, 2>(c, ap, sp) : launch_adaptive<float, 1>(c, ap, sp);
    if (rc) return rc;
    c->counters_pending = true;
    c->counters_counted = true;
  }

  c->last_path = !adaptive ? BEMCUB_PATH_FIXED : paired ? BEMCUB_PATH_PAIRED : BEMCUB_PATH_ADAPTIVE;
  c->stats.field_points_per_lane = sp.R;
  c->last_ipi = precision != BEMCUB_F64 ? 0 : grad ? 28 : out_E ? 18 : 12;
  mark(c, 2);
  // a6: cross-split reduction and the 1/(4 pi eps0) prefactor
  const int threads = 256;
  reduce_scale_kernel<<<(unsigned)((m + threads - 1) / threads), threads, 0, c->stream>>>(
      m, sp.nsplit, m, (const double4*)c->partial.ptr, (const double*)c->partial_g.ptr, coulomb_k(), perm, out_phi, out_E, out_G);
  count_launch(c);
  CUDA_TRY(cudaGetLastError());
  mark(c, 3);
  c->timing_valid = c->timing;
  return BEMCUB_OK;
}

}  // namespace

extern "C" {

int bemcub_eval(bemcub_ctx* c, const double* sigma, int rule_id, const bemcub_policy* host_policy, int64_t m,
                const double* field_pts, double* out_phi, double* out_E, int precision) {
  return eval_common(c, sigma, rule_id, host_policy, m, field_pts, out_phi, out_E, nullptr, precision);
}

int bemcub_eval_linear(bemcub_ctx* c, const double* sigma_vertex, int rule_id, const bemcub_policy* host_policy, int64_t m,
                       const double* field_pts, double* out_phi, double* out_E, int precision) {
  if (c && c->n > 0 && !sigma_vertex) return BEMCUB_ERR_INVALID_ARG;
  return eval_common(c, nullptr, rule_id, host_policy, m, field_pts, out_phi, out_E, nullptr, precision, false, sigma_vertex);
}

int bemcub_eval_pairs(bemcub_ctx* c, int64_t npairs, const uint8_t* type, const double* verts, const double* sigma, int method,
                      const bemcub_policy* host_policy, const double* field_pts, double* out_phi, double* out_E, int precision) {
  if (!c || npairs < 0) return BEMCUB_ERR_INVALID_ARG;
  if (!((method >= -1 && method <= BEMCUB_METHOD_ANALYTIC) || (method >= BEMCUB_METHOD_DUFFY_L0 && method <= BEMCUB_METHOD_DUFFY_L0 + 4)))
    return BEMCUB_ERR_BAD_RULE;
  if (precision != BEMCUB_F64 && precision != BEMCUB_F32) return BEMCUB_ERR_INVALID_ARG;
  PairsParams pp;
  if (method == BEMCUB_RULE_ADAPTIVE) {
    int rc = build_policy(host_policy, &pp.pol);
    if (rc) return rc;
  }
  if (npairs == 0) return BEMCUB_OK;
  if (!type || !verts || !field_pts || !out_phi) return BEMCUB_ERR_INVALID_ARG;
  DeviceGuard g(c->device);
  pp.K = npairs;
  pp.type = type;
  pp.verts = verts;
  pp.sigma = sigma;
  pp.method = method;
  pp.field = field_pts;
  pp.phi = out_phi;
  pp.E = out_E;
  pp.k = coulomb_k();
  const int threads = 128;
  const unsigned blocks = (unsigned)((npairs + threads - 1) / threads);
  if (precision == BEMCUB_F64) eval_pairs_kernel<double><<<blocks, threads, 0, c->stream>>>(pp);
  else eval_pairs_kernel<float><<<blocks, threads, 0, c->stream>>>(pp);
  c->stats.kernel_launches += 1;
  c->stats.last_eval_launches = 1;
  CUDA_TRY(cudaGetLastError());
  return BEMCUB_OK;
}

int bemcub_eval_gradient(bemcub_ctx* c, const double* sigma, int rule_id, const bemcub_policy* host_policy, int64_t m,
                         const double* field_pts, double* out_phi, double* out_E, double* out_G) {
  if (!out_G) return BEMCUB_ERR_INVALID_ARG;
  return eval_common(c, sigma, rule_id, host_policy, m, field_pts, out_phi, out_E, out_G, BEMCUB_F64);
}

}  // extern "C"

#include "bemcub_solve.inl"

extern "C" {

int bemcub_assemble_rows(bemcub_ctx* c, const bemcub_policy* host_policy, int64_t row0, int64_t nrows, double* out_rows,
                         int64_t ld) {
  if (!c) return BEMCUB_ERR_INVALID_ARG;
  if (!c->has_mesh) return BEMCUB_ERR_NO_ELEMENTS;
  if (row0 < 0 || nrows < 0 || row0 + nrows > c->n || ld < c->n) return BEMCUB_ERR_INVALID_ARG;
  if (c->n > kAsmMaxN) return BEMCUB_ERR_TOO_MANY_ELEMENTS;  // the kernel's near-pair queue packs the column into 25 bits
  PolicyDev pol;
  int rc = build_policy(host_policy, &pol);
  if (rc) return rc;
  if (nrows == 0 || c->n == 0) return BEMCUB_OK;
  if (!out_rows) return BEMCUB_ERR_INVALID_ARG;
  DeviceGuard g(c->device);
  c->stats.last_eval_launches = 0;
  c->timing_valid = false;
  mark(c, 0);
  AssembleParams ap;
  for (int l = 0; l < 5; ++l) {
    bool used = false;
    for (int w = 0; w <= 5; ++w) used |= (pol.map[w] == l);
    if (used) c->charged64[l] = false;
    // unit sigma; every element padded to a multiple of kAsmU points (zero charges): the fill kernel
    // takes kAsmU points per trip and has no remainder loop
    ap.stride[l] = (c->stride[l] + kAsmU - 1) / kAsmU * kAsmU;
    if (used && (rc = expand_level<double>(c, l, nullptr, c->pts64[l], nullptr, ap.stride[l], coulomb_k()))) return rc;
    ap.lvl_pts[l] = (const double4*)c->pts64[l].ptr;
  }
  // A tile is 128 consecutive rows and its row groups 32: they have to be compact patches whatever the
  // order the caller's elements come in (a shuffled level-5 icosphere otherwise executes 33 points for
  // every entry: 12.1 instead of 5.3 ms).  So the centroids are put in Morton order - the sort of step a2
  // (kernels_sort.cuh), once per mesh and row window - and the rows are taken in that order where it gives
  // clearly tighter 32-row groups than the caller's own (a device flag: no host round trip).
  ap.row_perm = nullptr;
  ap.use_perm = nullptr;
  if (nrows > kAsmRows && nrows < ((int64_t)1 << 31)) {
    if (c->asm_perm_row0 != row0 || c->asm_perm_nrows != nrows) {
      c->asm_perm_row0 = c->asm_perm_nrows = -1;
      if ((rc = ensure(c->asm_cen, (size_t)nrows * 24)) || (rc = ensure(c->asm_perm, (size_t)nrows * 4 + 32))) return rc;
      CUDA_TRY(cudaMemcpy2DAsync(c->asm_cen.ptr, 24, (const double4*)c->cenL.ptr + row0, 32, 24, (size_t)nrows,
                                 cudaMemcpyDeviceToDevice, c->stream));
      const uint32_t* perm = nullptr;
      const double* sorted = nullptr;
      c->sort_perm = nullptr;  // the sort buffers are shared with the evaluation calls
      if ((rc = sort_field_points(c, nrows, (const double*)c->asm_cen.ptr, &perm, &sorted))) return rc;
      CUDA_TRY(cudaMemcpyAsync(c->asm_perm.ptr, perm, (size_t)nrows * 4, cudaMemcpyDeviceToDevice, c->stream));
      const int64_t ngroups = (nrows + 31) / 32;
      float* radius = (float*)c->asm_cen.ptr;  // the packed centroids have served the sort
      int* flag = (int*)((char*)c->asm_perm.ptr + (((size_t)nrows * 4 + 15) & ~(size_t)15));
      group_radius_kernel<<<(unsigned)((2 * ngroups * 32 + 255) / 256), 256, 0, c->stream>>>(
          nrows, (const double4*)c->cenL.ptr + row0, (const uint32_t*)c->asm_perm.ptr, ngroups, radius);
      choose_row_order_kernel<<<1, 32, 0, c->stream>>>(ngroups, radius, flag);
      count_launch(c, 2);
      CUDA_TRY(cudaGetLastError());
      c->asm_perm_row0 = row0;
      c->asm_perm_nrows = nrows;
    }
    ap.row_perm = (const uint32_t*)c->asm_perm.ptr;
    ap.use_perm = (const int*)((const char*)c->asm_perm.ptr + (((size_t)nrows * 4 + 15) & ~(size_t)15));
  }
  ap.cenL = (const double4*)c->cenL.ptr;
  ap.type = (const uint8_t*)c->type.ptr;
  ap.verts = (const double*)c->verts.ptr;
  ap.n = c->n;
  ap.pol = pol;
  ap.row0 = row0;
  ap.nrows = nrows;
  ap.out = out_rows;
  ap.ld = ld;
  ap.k = coulomb_k();
  ap.counters = c->d_counters;
  ap.queue = c->d_counters + 2;
  CUDA_TRY(cudaMemsetAsync(c->d_counters, 0, 8 * sizeof(unsigned long long), c->stream));
  // items = (128-row tile) x (split of the columns, a multiple of 32): about 16 per warp, each met twice - the kernel
  // runs the queue once for the expensive column batches of every item and once for the cheap ones (measured on
  // config 3: 8 - 16 items per warp 5.25 ms, 32: 5.39, 64: 5.58, 4: 5.44; one pass over the queue: 5.33 ms at best)
  const int64_t warps = (int64_t)c->num_sms * kAsmWarps;
  ap.nrowtiles = (nrows + kAsmRows - 1) / kAsmRows;
  const int64_t batches = (c->n + 31) / 32;
  int64_t nsplit = std::max<int64_t>(1, std::min<int64_t>(batches, (16 * warps + ap.nrowtiles - 1) / ap.nrowtiles));
  ap.cols_per_split = ((batches + nsplit - 1) / nsplit) * 32;
  nsplit = (c->n + ap.cols_per_split - 1) / ap.cols_per_split;
  ap.nitems = ap.nrowtiles * nsplit;
  const int grid = (int)std::min<int64_t>(c->num_sms, (ap.nitems + kAsmWarps - 1) / kAsmWarps);
  mark(c, 1);
  assemble_kernel<<<grid, kAsmThreads, assemble_smem_bytes(), c->stream>>>(ap);
  c->last_ipi = 12;
  count_launch(c);
  CUDA_TRY(cudaGetLastError());
  mark(c, 2);
  mark(c, 3);
  c->timing_valid = c->timing;
  c->counters_pending = true;
  c->counters_counted = true;
  return BEMCUB_OK;
}

int bemcub_assemble(bemcub_ctx* c, const bemcub_policy* host_policy, double* out_matrix, int64_t ld) {
  if (!c) return BEMCUB_ERR_INVALID_ARG;
  if (!c->has_mesh) return BEMCUB_ERR_NO_ELEMENTS;
  return bemcub_assemble_rows(c, host_policy, 0, c->n, out_matrix, ld);
}

int bemcub_set_elements_host(bemcub_ctx* c, int64_t n, const uint8_t* host_type, const double* host_verts) {
  if (!c || n < 0 || (n > 0 && (!host_type || !host_verts))) return BEMCUB_ERR_INVALID_ARG;
  DeviceGuard g(c->device);
  int rc;
  const size_t nn = (size_t)std::max<int64_t>(n, 1);
  if ((rc = ensure(c->host_stage[0], nn)) || (rc = ensure(c->host_stage[1], nn * 72))) return rc;
  if (n > 0) {
    CUDA_TRY(cudaMemcpyAsync(c->host_stage[0].ptr, host_type, (size_t)n, cudaMemcpyHostToDevice, c->stream));
    CUDA_TRY(cudaMemcpyAsync(c->host_stage[1].ptr, host_verts, (size_t)n * 72, cudaMemcpyHostToDevice, c->stream));
  }
  return bemcub_set_elements(c, n, (const uint8_t*)c->host_stage[0].ptr, (const double*)c->host_stage[1].ptr);
}

int bemcub_eval_host(bemcub_ctx* c, const double* host_sigma, int rule_id, const bemcub_policy* host_policy, int64_t m,
                     const double* host_field_pts, double* host_phi, double* host_E, int precision) {
  if (!c || m < 0) return BEMCUB_ERR_INVALID_ARG;
  if (!c->has_mesh) return BEMCUB_ERR_NO_ELEMENTS;
  if (m == 0) return BEMCUB_OK;
  if (!host_field_pts || (!host_phi && !host_E) || (c->n > 0 && !host_sigma)) return BEMCUB_ERR_INVALID_ARG;
  DeviceGuard g(c->device);
  int rc;
  const size_t nn = (size_t)std::max<int64_t>(c->n, 1);
  if ((rc = ensure(c->host_stage[2], nn * 8)) || (rc = ensure(c->host_stage[3], (size_t)m * 24)) ||
      (rc = ensure(c->host_stage[4], (size_t)m * 32)))
    return rc;
  double* d_sigma = (double*)c->host_stage[2].ptr;
  double* d_pts = (double*)c->host_stage[3].ptr;
  double* d_phi = (double*)c->host_stage[4].ptr;
  double* d_E = d_phi + m;
  if (c->n > 0) CUDA_TRY(cudaMemcpyAsync(d_sigma, host_sigma, (size_t)c->n * 8, cudaMemcpyHostToDevice, c->stream));
  CUDA_TRY(cudaMemcpyAsync(d_pts, host_field_pts, (size_t)m * 24, cudaMemcpyHostToDevice, c->stream));
  rc = bemcub_eval(c, d_sigma, rule_id, host_policy, m, d_pts, host_phi ? d_phi : nullptr, host_E ? d_E : nullptr, precision);
  if (rc) return rc;
  if (host_phi) CUDA_TRY(cudaMemcpyAsync(host_phi, d_phi, (size_t)m * 8, cudaMemcpyDeviceToHost, c->stream));
  if (host_E) CUDA_TRY(cudaMemcpyAsync(host_E, d_E, (size_t)m * 24, cudaMemcpyDeviceToHost, c->stream));
  CUDA_TRY(cudaStreamSynchronize(c->stream));
  return BEMCUB_OK;
}

int bemcub_fp64_issue_sweep(bemcub_ctx* c, double seconds_per_variant, double* host_rates, double* host_sm_mhz) {
  if (!c || !host_rates || !(seconds_per_variant > 0.0) || seconds_per_variant > 10.0) return BEMCUB_ERR_INVALID_ARG;
  DeviceGuard g(c->device);
  const int threads = 256;
  int rc = ensure(c->partial, (size_t)threads * c->num_sms * 4 * 8);
  if (rc) return rc;
  cudaEvent_t e0, e1;
  CUDA_TRY(cudaEventCreate(&e0));
  CUDA_TRY(cudaEventCreate(&e1));
  unsigned long long* clk = c->d_counters + 6;
  auto run = [&](int mix, int blocks, int iters, float* ms) -> int {
    CUDA_TRY(cudaEventRecord(e0, c->stream));
    double* out = (double*)c->partial.ptr;
    switch (mix) {
      case 0: fp64_issue_kernel<0><<<blocks, threads, 0, c->stream>>>(out, clk, iters, 0.999999, 1e-9, 3); break;
      case 1: fp64_issue_kernel<1><<<blocks, threads, 0, c->stream>>>(out, clk, iters, 0.999999, 1e-9, 3); break;
      case 2: fp64_issue_kernel<2><<<blocks, threads, 0, c->stream>>>(out, clk, iters, 0.999999, 1e-9, 3); break;
      case 3: fp64_issue_kernel<3><<<blocks, threads, 0, c->stream>>>(out, clk, iters, 0.999999, 1e-9, 3); break;
      case 4: fp64_issue_kernel<4><<<blocks, threads, 0, c->stream>>>(out, clk, iters, 0.999999, 1e-9, 3); break;
      default: fp64_issue_kernel<5><<<blocks, threads, 0, c->stream>>>(out, clk, iters, 0.999999, 1e-9, 3); break;
    }
    c->stats.kernel_launches += 1;
    CUDA_TRY(cudaGetLastError());
    CUDA_TRY(cudaEventRecord(e1, c->stream));
    CUDA_TRY(cudaEventSynchronize(e1));
    CUDA_TRY(cudaEventElapsedTime(ms, e0, e1));
    return BEMCUB_OK;
  };
  for (int mix = 0; mix < BEMCUB_PEAK_VARIANTS / 3; ++mix) {
    const int chains = mix == 3 ? 18 : 16;
    for (int occ = 0; occ < 3; ++occ) {
      const int per_sm = 1 << occ;  // CTAs of 8 warps per SM: 8, 16, 32 warps
      const int blocks = c->num_sms * per_sm;
      const double per_iter = 4.0 * chains * threads * blocks;  // FP64 lane-instructions per loop iteration of the grid
      float ms = 0.f;
      if ((rc = run(mix, blocks, 2000, &ms))) return rc;  // warm-up
      if ((rc = run(mix, blocks, 20000, &ms))) return rc;  // calibration
      const double rate0 = per_iter * 20000 / (ms * 1e-3);
      // one launch of the requested length: the sustained rate, with the clock it was sustained at
      const int iters = (int)std::min(2.0e9, std::max(1000.0, seconds_per_variant * rate0 / per_iter));
      if ((rc = run(mix, blocks, iters, &ms))) return rc;
      host_rates[mix * 3 + occ] = per_iter * iters / (ms * 1e-3);
      if (host_sm_mhz) {
        unsigned long long h[2] = {0, 0};
        CUDA_TRY(cudaMemcpy(h, clk, sizeof(h), cudaMemcpyDeviceToHost));
        host_sm_mhz[mix * 3 + occ] = h[1] ? 1e3 * (double)h[0] / (double)h[1] : 0.0;
      }
    }
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  return BEMCUB_OK;
}

int bemcub_fp64_peak(bemcub_ctx* c, double seconds, double* host_fp64_inst_per_s) {
  if (!c || !host_fp64_inst_per_s || !(seconds > 0.0) || seconds > 30.0) return BEMCUB_ERR_INVALID_ARG;
  double rates[BEMCUB_PEAK_VARIANTS];
  int rc = bemcub_fp64_issue_sweep(c, seconds / BEMCUB_PEAK_VARIANTS, rates, nullptr);
  if (rc) return rc;
  *host_fp64_inst_per_s = *std::max_element(rates, rates + BEMCUB_PEAK_VARIANTS);
  return BEMCUB_OK;
}

int bemcub_inner_loop_rate(bemcub_ctx* c, double seconds, double* host_interactions_per_s) {
  if (!c || !host_interactions_per_s || !(seconds > 0.0) || seconds > 30.0) return BEMCUB_ERR_INVALID_ARG;
  DeviceGuard g(c->device);
  constexpr int R = 4;
  const int64_t npts_field = (int64_t)c->num_sms * kWarpsPerCta * 32 * R;
  int rc;
  if ((rc = ensure(c->partial, (size_t)npts_field * 32)) || (rc = ensure(c->host_stage[3], (size_t)npts_field * 24)) ||
      (rc = ensure(c->host_stage[4], (size_t)kStages * kBuf * 32)))
    return rc;
  // synthetic resident data: source points in the unit cube, field points 3..4 away
  fill_synthetic_kernel<<<(unsigned)((npts_field + 255) / 256), 256, 0, c->stream>>>(
      npts_field, (double*)c->host_stage[3].ptr, kStages * kBuf, (double4*)c->host_stage[4].ptr);
  c->stats.kernel_launches += 1;
  const size_t smem = eval_smem_bytes<double>();
  cudaEvent_t e0, e1;
  CUDA_TRY(cudaEventCreate(&e0));
  CUDA_TRY(cudaEventCreate(&e1));
  const int cnt = kBuf - 16;  // a typical adaptive stage: 112 points
  auto run = [&](int trips, float* ms) -> int {
    CUDA_TRY(cudaEventRecord(e0, c->stream));
    inner_loop_kernel<R><<<c->num_sms, kThreads, smem, c->stream>>>((const double4*)c->host_stage[4].ptr,
                                                                   (const double*)c->host_stage[3].ptr, cnt, trips,
                                                                   (double4*)c->partial.ptr);
    c->stats.kernel_launches += 1;
    CUDA_TRY(cudaGetLastError());
    CUDA_TRY(cudaEventRecord(e1, c->stream));
    CUDA_TRY(cudaEventSynchronize(e1));
    CUDA_TRY(cudaEventElapsedTime(ms, e0, e1));
    return BEMCUB_OK;
  };
  const double per_trip = (double)npts_field * cnt;
  float ms = 0.f;
  if ((rc = run(200, &ms))) return rc;
  if ((rc = run(2000, &ms))) return rc;
  const double rate0 = per_trip * 2000 / (ms * 1e-3);
  const int trips = (int)std::min(2.0e9, std::max(100.0, 0.25 * rate0 / per_trip));
  double total_ms = 0.0, total = 0.0;
  while (total_ms < seconds * 1e3) {
    if ((rc = run(trips, &ms))) return rc;
    total_ms += ms;
    total += per_trip * trips;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  *host_interactions_per_s = total / (total_ms * 1e-3);
  return BEMCUB_OK;
}

int bemcub_get_stats(bemcub_ctx* c, bemcub_stats* host_stats) {
  if (!c || !host_stats) return BEMCUB_ERR_INVALID_ARG;
  DeviceGuard g(c->device);
  refresh_counters(c);
  *host_stats = c->stats;
  return BEMCUB_OK;
}

int bemcub_set_timing(bemcub_ctx* c, int enable) {
  if (!c) return BEMCUB_ERR_INVALID_ARG;
  DeviceGuard g(c->device);
  if (enable)
    for (int i = 0; i < 4; ++i)
      if (!c->ev[i]) CUDA_TRY(cudaEventCreate(&c->ev[i]));
  c->timing = enable != 0;
  c->timing_valid = false;
  return BEMCUB_OK;
}

int bemcub_get_timing(bemcub_ctx* c, double* host_ms_total, double* host_ms_kernel) {
  if (!c) return BEMCUB_ERR_INVALID_ARG;
  if (!c->timing_valid) return BEMCUB_ERR_INVALID_ARG;
  DeviceGuard g(c->device);
  CUDA_TRY(cudaEventSynchronize(c->ev[3]));
  float a = 0.f, b = 0.f;
  CUDA_TRY(cudaEventElapsedTime(&a, c->ev[0], c->ev[3]));
  CUDA_TRY(cudaEventElapsedTime(&b, c->ev[1], c->ev[2]));
  if (host_ms_total) *host_ms_total = a;
  if (host_ms_kernel) *host_ms_kernel = b;
  return BEMCUB_OK;
}

int bemcub_last_path(bemcub_ctx* c, int* host_path) {
  if (!c || !host_path) return BEMCUB_ERR_INVALID_ARG;
  *host_path = c->last_path;
  return BEMCUB_OK;
}

int bemcub_reset_stats(bemcub_ctx* c) {
  if (!c) return BEMCUB_ERR_INVALID_ARG;
  c->stats = bemcub_stats{};
  c->counters_pending = false;
  return BEMCUB_OK;
}

}  // extern "C"

// ------------------------------------------------------------------------------------------------
// bemcub_eval_few_noalloc (include/bemcub.h): the few-point evaluation for callers that must not
// allocate.  eval_few_kernel needs two pieces of global scratch - the CTAs' partial sums and the
// counters by which the last CTA of a pass knows it is the last - which bemcub_eval takes from
// ctx-owned cudaMalloc memory.  Here they live in the array below: part of the library's image, put
// on every GPU that loads the library and kept there until the process exits (about 641 KB each).
//   bytes [0, 512)      counters: interaction tallies, then one "CTAs done" counter per pass; the
//                       kernel counts up from zero, so they are cleared before every launch
//   bytes [512, end)    partial sums [CTA][m] (double4); every CTA writes all of its entries before
//                       the last one reads them, so what the previous call left there never matters
// The array is shared by every ctx and every stream of the process: two calls that are on the GPU
// at the same time would count in each other's counters and overwrite each other's sums.
constexpr int kNoAllocMaxM = kFewMaxM;  // 64 field points per call
constexpr int kNoAllocMaxCtas = 320;    // two CTAs per SM, as bemcub_eval launches them: devices of up to 160 SMs
constexpr size_t kNoAllocCounterBytes = 512;
constexpr size_t kNoAllocBytes = kNoAllocCounterBytes + (size_t)kNoAllocMaxCtas * kNoAllocMaxM * sizeof(double4);
static_assert(kCounterSlots * sizeof(unsigned long long) <= kNoAllocCounterBytes, "counter block too small");
static __device__ __align__(256) unsigned char g_noalloc_scratch[kNoAllocBytes];

namespace {

// In host code `g_noalloc_scratch` is only a handle for the runtime, not somewhere a kernel can write:
// the array's address on a given GPU comes from cudaGetSymbolAddress, asked once per device with that
// device current, and that address is what the kernel gets.
constexpr int kNoAllocMaxDevices = 64;
void* g_noalloc_addr[kNoAllocMaxDevices] = {};
std::mutex g_noalloc_mutex;

int noalloc_scratch_of_current_device(int device, unsigned char** out) {
  if (device < 0 || device >= kNoAllocMaxDevices) return BEMCUB_ERR_INVALID_ARG;
  std::lock_guard<std::mutex> lock(g_noalloc_mutex);
  if (!g_noalloc_addr[device]) {
    void* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
    if (e != cudaSuccess || !p) {
      cudaGetLastError();
      return BEMCUB_ERR_CUDA;
    }
    g_noalloc_addr[device] = p;
  }
  *out = static_cast<unsigned char*>(g_noalloc_addr[device]);
  return BEMCUB_OK;
}

}  // namespace

extern "C" int bemcub_eval_few_noalloc(bemcub_ctx* c, const double* sigma, int rule_id, const bemcub_policy* host_policy,
                                       int64_t m, const double* field_pts, double* out_phi, double* out_E) {
  if (!c || m < 0) return BEMCUB_ERR_INVALID_ARG;
  if (!c->has_mesh) return BEMCUB_ERR_NO_ELEMENTS;
  if (rule_id < -1 || rule_id > 4) return BEMCUB_ERR_BAD_RULE;
  const bool adaptive = rule_id == BEMCUB_RULE_ADAPTIVE;
  PolicyDev pol;
  if (adaptive) {
    const int rc = build_policy(host_policy, &pol);
    if (rc) return rc;
  }
  if (m == 0) return BEMCUB_OK;
  const int blocks = c->num_sms * 2;  // the grid of bemcub_eval's few-point route: same sums in the same order
  if (m > kNoAllocMaxM || blocks > kNoAllocMaxCtas) return BEMCUB_ERR_FIXED_SCRATCH;
  if (!field_pts || !out_phi || (c->n > 0 && !sigma)) return BEMCUB_ERR_INVALID_ARG;
  DeviceGuard g(c->device);
  if (!g.ok) return BEMCUB_ERR_CUDA;
  if (c->n == 0) {  // empty mesh: zero potential and field
    CUDA_TRY(cudaMemsetAsync(out_phi, 0, (size_t)m * 8, c->stream));
    if (out_E) CUDA_TRY(cudaMemsetAsync(out_E, 0, (size_t)m * 24, c->stream));
    return BEMCUB_OK;
  }
  unsigned char* scratch = nullptr;
  const int rc = noalloc_scratch_of_current_device(c->device, &scratch);
  if (rc) return rc;

  FewParams fw;
  fw.cenL = (const double4*)c->cenL.ptr;
  fw.type = (const uint8_t*)c->type.ptr;
  fw.verts = (const double*)c->verts.ptr;
  fw.sigma = sigma;  // read in place: nothing of this call is kept in the ctx
  fw.n = c->n;
  if (adaptive) fw.pol = pol;
  fw.rule = adaptive ? -1 : rule_id;
  fw.field = field_pts;
  fw.m = m;
  fw.counters = reinterpret_cast<unsigned long long*>(scratch);
  fw.done = reinterpret_cast<unsigned*>(fw.counters + 8);
  fw.partial = reinterpret_cast<double4*>(scratch + kNoAllocCounterBytes);
  fw.area = (const double*)c->area.ptr;
  fw.sigma_v = nullptr;
  fw.k = coulomb_k();
  fw.out_phi = out_phi;
  fw.out_E = out_E;
  CUDA_TRY(cudaMemsetAsync(scratch, 0, kNoAllocCounterBytes, c->stream));
  const int per_pass = m >= 3 ? kFewM : (int)m;
  const dim3 grid((unsigned)blocks, (unsigned)((m + per_pass - 1) / per_pass));
  const int threads = kFewWarps * 32;
  if (out_E) {
    if (per_pass == 1) eval_few_kernel<kModePhiE, 1><<<grid, threads, 0, c->stream>>>(fw);
    else if (per_pass == 2) eval_few_kernel<kModePhiE, 2><<<grid, threads, 0, c->stream>>>(fw);
    else eval_few_kernel<kModePhiE, kFewM><<<grid, threads, 0, c->stream>>>(fw);
  } else {
    if (per_pass == 1) eval_few_kernel<kModePhi, 1><<<grid, threads, 0, c->stream>>>(fw);
    else if (per_pass == 2) eval_few_kernel<kModePhi, 2><<<grid, threads, 0, c->stream>>>(fw);
    else eval_few_kernel<kModePhi, kFewM><<<grid, threads, 0, c->stream>>>(fw);
  }
  c->stats.kernel_launches += 1;
  CUDA_TRY(cudaGetLastError());
  return BEMCUB_OK;
}
