// common.cuh -- device helpers shared by the librfim kernels (sm_100a).
//
// Exact integer form of the sigma cut for uint8 data (include/rfim.h, DESIGN.md "Exact integer
// evaluation"): with S = sum x, Q = sum x^2 over the N snapshot values, V = N Q - S^2 and the
// threshold k = p / 2^16,
//     |x - S/N| > k sqrt(V)/N   <=>   (N x - S)^2 > floor(p^2 V / 2^32) =: W
// (the left side is an integer, so flooring the right side keeps the test exact).  Because the
// decision depends only on the value x, one cut collapses to two byte bounds: the kept values are
// the interval lo <= x <= hi (empty: lo = 1, hi = 0).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

namespace rfim {

constexpr unsigned FULL = 0xffffffffu;

struct U8Cut {
  uint32_t N;
  uint32_t S;      // < 2^32 because N <= 2^24
  uint64_t W;      // low 64 bits of floor(p^2 V / 2^32)
  bool never;      // W >= 2^64: no deviation can exceed it
};

// V = N Q - S^2 = N^2 * variance (< 2^62 for N <= 2^24)
__device__ __forceinline__ U8Cut make_cut_u8(uint32_t N, uint64_t S, uint64_t V, uint32_t p) {
  U8Cut c;
  const uint64_t p2 = (uint64_t)p * p;                  // < 2^48
  const uint64_t hi = __umul64hi(p2, V), lo = p2 * V;   // 128-bit product p^2 V
  c.N = N;
  c.S = (uint32_t)S;
  c.W = (hi << 32) | (lo >> 32);
  c.never = (hi >> 32) != 0;
  return c;
}

// true <=> value x is cut (|t_i - mu| > n sigma, strict, two-sided)
__device__ __forceinline__ bool cut_flags_u8(const U8Cut& c, uint32_t x) {
  const int64_t d = (int64_t)((uint64_t)c.N * x) - (int64_t)c.S;   // |d| < 2^32
  const uint32_t ad = (uint32_t)(d < 0 ? -d : d);
  const uint64_t d2 = (uint64_t)ad * ad;
  return !c.never && d2 > c.W;
}

// replacement mean for integers, round half up: floor((2S + N) / (2N))   (always in 0..255)
__device__ __forceinline__ uint32_t rounded_mean_u8(uint32_t N, uint64_t S) {
  const uint64_t a = 2 * S + N, b = 2 * (uint64_t)N;      // a < 2^33, b <= 2^25, quotient <= 255
  uint32_t r = (uint32_t)__fdividef((float)a, (float)b);  // within 1 of the quotient
  if (r > 255u) r = 255u;
  if (a < (1ull << 31)) {                                 // 32-bit arithmetic: r b <= a + b < 2^32
    const uint32_t a32 = (uint32_t)a, b32 = (uint32_t)b;
    while (r * b32 > a32) --r;
    while (a32 - r * b32 >= b32) ++r;
    return r;
  }
  while ((uint64_t)r * b > a) --r;
  while (a - (uint64_t)r * b >= b) ++r;
  return r;
}

// Kept interval [lo, hi] of byte values for one cut, evaluated by a whole warp: lane l tests the
// eight values 8l .. 8l+7 with the exact predicate.  All lanes return the same lo, hi.
__device__ __forceinline__ void warp_bounds_u8(const U8Cut& c, int lane, int& lo, int& hi) {
  uint32_t m = 0;
#pragma unroll
  for (int j = 0; j < 8; ++j) m |= (cut_flags_u8(c, (uint32_t)(lane * 8 + j)) ? 0u : 1u) << j;
  const uint32_t any = __ballot_sync(FULL, m != 0);
  if (any == 0) { lo = 1; hi = 0; return; }
  const int l0 = __ffs(any) - 1, l1 = 31 - __clz(any);
  const uint32_t m0 = __shfl_sync(FULL, m, l0), m1 = __shfl_sync(FULL, m, l1);
  lo = l0 * 8 + __ffs(m0) - 1;
  hi = l1 * 8 + (31 - __clz(m1));
}

// Same interval for ONE thread (used where threads own columns): the kept set, if not empty,
// contains floor(S/N) or floor(S/N)+1; binary search outward on the monotone predicate.
__device__ __forceinline__ void thread_bounds_u8(const U8Cut& c, int& lo, int& hi) {
  uint32_t x0 = (uint32_t)__fdividef((float)c.S, (float)c.N);
  while ((uint64_t)(x0 + 1) * c.N <= c.S) ++x0;
  while ((uint64_t)x0 * c.N > c.S) --x0;                     // x0 = floor(S/N) <= 255
  int mid;
  if (!cut_flags_u8(c, x0)) mid = (int)x0;
  else if (x0 < 255 && !cut_flags_u8(c, x0 + 1)) mid = (int)x0 + 1;
  else { lo = 1; hi = 0; return; }
  int a = 0, b = mid;                                        // smallest kept value in [0, mid]
  while (a < b) { int m = (a + b) >> 1; if (cut_flags_u8(c, (uint32_t)m)) a = m + 1; else b = m; }
  lo = a;
  a = mid; b = 255;                                          // largest kept value in [mid, 255]
  while (a < b) { int m = (a + b + 1) >> 1; if (cut_flags_u8(c, (uint32_t)m)) b = m - 1; else a = m; }
  hi = a;
}

// Same interval for ONE thread in closed form: with T = isqrt(W) (floor), |N x - S| <= T <=> (N x - S)^2 <= W,
// so the kept values are ceil((S - T) / N) <= x <= floor((S + T) / N), clamped to 0..255.  The square root is
// taken in fp64 and corrected with exact integer checks; the quotients are float estimates corrected the same
// way.  Result identical to warp_bounds_u8 (empty interval: lo = 1, hi = 0).
__device__ __forceinline__ uint32_t div_floor_u64(uint64_t a, uint32_t n) {   // a / n, quotient < 2^24 * 512
  uint64_t q = (uint64_t)__fdividef((float)a, (float)n);
  while (q * n > a) --q;
  while (a - q * n >= n) ++q;
  return (uint32_t)q;
}
__device__ __forceinline__ void thread_bounds_u8_sqrt(const U8Cut& c, int& lo, int& hi) {
  if (c.never) { lo = 0; hi = 255; return; }
  uint64_t T = (uint64_t)__dsqrt_rd((double)c.W);              // within 1 of floor(sqrt(W)), below 2^32
  if (T > 0xffffffffull) T = 0xffffffffull;
  while (T * T > c.W) --T;
  while (T < 0xffffffffull && (T + 1) * (T + 1) <= c.W) ++T;
  const uint64_t S = c.S, N = c.N;
  const uint64_t top = S + T;                                  // < 2^33
  const uint64_t hq = top >= 256ull * N ? 255ull : div_floor_u64(top, c.N);
  hi = (int)(hq > 255ull ? 255ull : hq);
  lo = S > T ? (int)div_floor_u64(S - T + N - 1, c.N) : 0;     // ceil((S - T) / N), <= 255 because S <= 255 N
  if (lo > hi) { lo = 1; hi = 0; }
}

// The same closed form with 32-bit quotients: floor(a / n) for a < 2^32 from inv = ceil(2^32 / n) is
// umulhi(a, inv) or one less (a inv / 2^32 < a / n + 1), so one exact check finishes it.  Used where n is the
// same for every column (FDSC: n = channels) and the host passes inv.
__device__ __forceinline__ uint32_t div_floor_u32(uint32_t a, uint32_t n, uint32_t inv) {
  uint32_t q = __umulhi(a, inv);
  if ((uint64_t)q * n > a) --q;
  return q;
}
// requires 2 <= n and S + T < 2^32 (else the caller uses thread_bounds_u8_sqrt); r = rounded mean floor((2S+n)/(2n))
__device__ __forceinline__ void thread_bounds_u8_sqrt32(const U8Cut& c, uint32_t inv, int& lo, int& hi, uint32_t& r) {
  const uint32_t S = c.S, N = c.N;
  r = div_floor_u32(S + (N >> 1), N, inv);                     // floor((2S+N)/(2N)) = floor((S + floor(N/2)) / N) for even N;
  if (N & 1u) {                                                // odd N: compare 2 (S - r N) + N with 2 N exactly
    const uint32_t rem2 = 2u * (S - div_floor_u32(S, N, inv) * N) + N;
    r = div_floor_u32(S, N, inv) + (rem2 >= 2u * N ? 1u : 0u);
  }
  if (c.never) { lo = 0; hi = 255; return; }
  uint64_t T = (uint64_t)__dsqrt_rd((double)c.W);
  if (T > 0xffffffffull) T = 0xffffffffull;
  while (T * T > c.W) --T;
  while (T < 0xffffffffull && (T + 1) * (T + 1) <= c.W) ++T;
  const uint64_t top = (uint64_t)S + T;
  if (top >= 256ull * N) hi = 255;
  else hi = (int)div_floor_u32((uint32_t)top, N, inv);         // top < 256 N <= 2^32
  lo = (uint64_t)S > T ? (int)div_floor_u32((uint32_t)(S - T) + N - 1u, N, inv) : 0;   // S - T + N - 1 < 2^32: S <= 255 N, N <= 2^24
  if (lo > hi) { lo = 1; hi = 0; }
}

__device__ __forceinline__ uint32_t warp_sum_u32(uint32_t v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(FULL, v, o);
  return v;
}
__device__ __forceinline__ uint64_t warp_sum_u64(uint64_t v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(FULL, v, o);
  return v;
}
__device__ __forceinline__ double warp_sum_f64(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(FULL, v, o);
  return v;
}

// ---------------------------------------------------------------- async-proxy (TMA bulk) wrappers
__device__ __forceinline__ uint32_t smem_addr(const void* p) {
  return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_addr(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_mbar_init() {
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_addr(bar)), "r"(bytes)
               : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_addr(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_LOOP:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra WAIT_DONE;\n"
      "bra WAIT_LOOP;\n"
      "WAIT_DONE:\n"
      "}\n" ::"r"(smem_addr(bar)),
      "r"(parity)
      : "memory");
}
// 1-D bulk copy global -> shared (16-byte aligned addresses, size a multiple of 16), completion on mbarrier
__device__ __forceinline__ void bulk_load(void* smem_dst, const void* gmem_src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   smem_addr(smem_dst)),
               "l"(gmem_src), "r"(bytes), "r"(smem_addr(bar))
               : "memory");
}
// L2 eviction policy for data that is touched once (a streamed row: read, or written, and never again)
__device__ __forceinline__ uint64_t l2_policy_evict_first() {
  uint64_t pol;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
  return pol;
}
// the same copies with an L2 cache hint
__device__ __forceinline__ void bulk_load_hint(void* smem_dst, const void* gmem_src, uint32_t bytes, uint64_t* bar,
                                               uint64_t policy) {
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(
          smem_addr(smem_dst)),
      "l"(gmem_src), "r"(bytes), "r"(smem_addr(bar)), "l"(policy)
      : "memory");
}
// 1-D bulk prefetch global -> L2 (16-byte aligned address, size a multiple of 16): no destination, nothing to wait for
__device__ __forceinline__ void bulk_prefetch_l2(const void* gmem_src, uint32_t bytes) {
  asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(gmem_src), "r"(bytes) : "memory");
}
// 1-D bulk copy shared -> global, tracked by bulk async-groups
__device__ __forceinline__ void bulk_store(void* gmem_dst, const void* smem_src, uint32_t bytes) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(gmem_dst),
               "r"(smem_addr(smem_src)), "r"(bytes)
               : "memory");
}
__device__ __forceinline__ void bulk_store_hint(void* gmem_dst, const void* smem_src, uint32_t bytes, uint64_t policy) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group.L2::cache_hint [%0], [%1], %2, %3;" ::"l"(gmem_dst),
               "r"(smem_addr(smem_src)), "r"(bytes), "l"(policy)
               : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void bulk_wait_read() {
  asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(N) : "memory");
}
template <int N>
__device__ __forceinline__ void bulk_wait_all() {
  asm volatile("cp.async.bulk.wait_group %0;" ::"n"(N) : "memory");
}
// generic-proxy writes to shared memory -> visible to the async proxy (before a bulk store)
__device__ __forceinline__ void fence_proxy_async_smem() {
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}

}  // namespace rfim
