// PTX wrappers and small device helpers shared by the bemcub kernels (sm_100a only).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace bemcub {

constexpr unsigned kFullMask = 0xffffffffu;

__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}

// ---- mbarrier + 1-D bulk TMA (cp.async.bulk, SASS UBLKCP) ------------------------------------
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() {
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
      "selp.u32 %0, 1, 0, p;\n"
      "}\n"
      : "=r"(ok)
      : "r"(bar), "r"(parity)
      : "memory");
  return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  while (!mbar_try_wait(bar, parity)) {
  }
}
// global -> shared bulk copy; bytes % 16 == 0, both addresses 16-byte aligned; completion is
// signalled on the mbarrier as `bytes` of transaction count.
__device__ __forceinline__ void tma_load_1d(uint32_t dst_smem, const void* src_gmem, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst_smem),
               "l"(src_gmem), "r"(bytes), "r"(bar)
               : "memory");
}

// ---- reciprocal square root ------------------------------------------------------------------
// What bounds the hot loops is the ISSUE port, not latency (profiles/r2_issue_model.md):
// an FP64 instruction holds a scheduler's dispatch for 2 cycles, 3 if it reads three distinct vector
// registers that are not in the operand-reuse cache, and every other instruction (MUFU, MOV, LDS,
// loop bookkeeping) takes a cycle of its own.  The refinement below is written for that model.
//
// MUFU.RSQ64H seed: reads only the high word of x and writes only the HIGH word of its result
// (~2^-20 relative error).  The PTX instruction returns the seed with a zero low word, which costs
// a MOV per call.  rsqrt_f64 instead takes the low word from `dead`, a value the caller does not
// need any more (an intermediate of x): ptxas then lets MUFU write into the high half of that
// value's register pair and the MOV disappears.  Any low word will do - it moves the seed by
// < 2^-20 of its value, which the correction below absorbs - and this one is a function of the
// interaction's own data, so results stay bit-reproducible.
__device__ __forceinline__ double rsqrt_seed(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  return y;
}
// 0.375 of the correction polynomial.  DFMA takes one immediate only (the 0.5), so this constant
// lives in a register; read from constant memory it cannot be re-materialised inside the loop
// (two MOVs per trip when written as a literal).
__constant__ double c_three_eighths = 0.375;

// ... and one third-order correction y = y0 (1 + e/2 + 3e^2/8), e = 1 - x y0^2 : 5 FP64 instructions,
// residual (5/16) e^3 < 2^-57 for |e| < 2^-18.  (A second-order step would leave ~4e-12: not enough
// for the 1e-12 parity bar nor for the paper's 1e-15 accuracy level.)  Written as
// y = fma(y0, e p, y0): two distinct registers, where fma(y0 e, p, y0) reads three.
__device__ __forceinline__ double rsqrt_f64(double x, double dead, double c375) {
  const double y0 = __hiloint2double(__double2hiint(rsqrt_seed(x)), __double2loint(dead));
  const double t = __dmul_rn(x, y0);
  const double e = __fma_rn(-t, y0, 1.0);
  const double p = __fma_rn(c375, e, 0.5);
  const double u = __dmul_rn(e, p);
  return __fma_rn(y0, u, y0);
}
__device__ __forceinline__ float rsqrt_f32(float x) {
  float y;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  // one Newton step: MUFU.RSQ is good to ~2^-22.4; this brings it to ~1 ulp of FP32
  const float e = fmaf(-x * y, y, 1.0f);
  return fmaf(0.5f * y, e, y);
}

// read-only 32-byte point record
__device__ __forceinline__ double4 ldg4(const double4* p) {
  const double2 a = __ldg(reinterpret_cast<const double2*>(p));
  const double2 b = __ldg(reinterpret_cast<const double2*>(p) + 1);
  return make_double4(a.x, a.y, b.x, b.y);
}

// ---- SM clock actually seen by a kernel ---------------------------------------------------------
// Thread 0 of CTA 0 (a persistent CTA lives as long as the launch) reads the SM cycle counter and the
// global nanosecond timer at both ends; counters[4] = cycles, counters[5] = ns.  cycles / ns is the
// clock the kernel really ran at - the denominator of the per-cycle roofline (bench.py).
__device__ __forceinline__ unsigned long long global_timer_ns() {
  unsigned long long t;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
  return t;
}
struct KernelClock {
  long long c0;
  unsigned long long t0;
  __device__ __forceinline__ void begin() {
    if (blockIdx.x == 0 && blockIdx.y == 0 && threadIdx.x == 0) {
      c0 = clock64();
      t0 = global_timer_ns();
    }
  }
  __device__ __forceinline__ void end(unsigned long long* counters) {
    if (counters && blockIdx.x == 0 && blockIdx.y == 0 && threadIdx.x == 0) {
      counters[4] = (unsigned long long)(clock64() - c0);
      counters[5] = global_timer_ns() - t0;
    }
  }
};

// ---- warp helpers ----------------------------------------------------------------------------
__device__ __forceinline__ double warp_min(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmin(v, __shfl_xor_sync(kFullMask, v, o));
  return v;
}
__device__ __forceinline__ double warp_max(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(kFullMask, v, o));
  return v;
}
// FP32 min / max over the warp with one REDUX each (order-preserving map to unsigned; no NaN expected)
__device__ __forceinline__ unsigned ordered_u32(float x) {
  const unsigned b = __float_as_uint(x);
  return (b >> 31) ? ~b : (b | 0x80000000u);
}
__device__ __forceinline__ float from_ordered_u32(unsigned u) { return __uint_as_float((u >> 31) ? (u & 0x7fffffffu) : ~u); }
__device__ __forceinline__ float warp_min_f32(float v) { return from_ordered_u32(__reduce_min_sync(kFullMask, ordered_u32(v))); }
__device__ __forceinline__ float warp_max_f32(float v) { return from_ordered_u32(__reduce_max_sync(kFullMask, ordered_u32(v))); }
__device__ __forceinline__ int warp_excl_scan(int v, int lane, int* total) {
  int x = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int y = __shfl_up_sync(kFullMask, x, o);
    if (lane >= o) x += y;
  }
  *total = __shfl_sync(kFullMask, x, 31);
  return x - v;
}

}  // namespace bemcub
