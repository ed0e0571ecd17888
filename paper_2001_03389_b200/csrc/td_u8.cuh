// td_u8.cuh -- time-domain sigma cut (TDSC, Fig. 2) for uint8 dynamic spectra.
//
// Two kernels:
//   td_u8_staged_kernel   the hot path.  One warp owns one
//       (beam, channel) row at a time.  T1: the row is brought into the warp's shared-memory slot
//       by one 1-D TMA bulk copy (cp.async.bulk, completion on an mbarrier); only the <= 15 head and
//       tail bytes that are not 16-byte aligned in global memory are moved by the lanes.  T2: exact
//       sum and sum of squares with IDP.4A over 16-byte groups.  T3: the cut collapses to two byte
//       bounds, found by evaluating the exact 64/128-bit predicate for all 256 byte values across the
//       warp.  T4: a packed range check (3 instructions per 32-bit word, VIADDMNMX.U16x2) finds the
//       16-byte groups that contain a value outside [lo, hi]; their indices are compacted into a
//       queue and only those groups are revisited byte by byte (replace, update S and Q
//       incrementally).  T5: next threshold, on chip.  T6: one TMA bulk store.  HBM sees one read
//       and one write per sample.
//   td_u8_generic_kernel  any alignment / stride / row length / window, mean or median: one CTA per
//       row, byte loads, iterations through global memory (L1/L2).  Correctness path, not tuned.
#pragma once

#include "common.cuh"

namespace rfim {

struct TdU8Params {
  const uint8_t* src;
  uint8_t* dst;
  int64_t rows;
  int64_t stride;
  int S;
  int window;                 // generic kernel only; >= 1
  int n_thr;
  int policy;                 // generic kernel only
  uint32_t p[16];             // thresholds as p / 2^16
  uint8_t* flags;             // optional [rows][S]
  unsigned long long* counts; // optional [n_thr]
  int slot_bytes;             // staged kernel: bytes per warp slot (multiple of 16)
  int queue_entries;          // staged kernel: u16 entries per warp queue
};

// ------------------------------------------------------------------------------------------------
// staged hot path
// ------------------------------------------------------------------------------------------------

// max over the 4 words of a group of ((v - LB) mod 2^16) for v in {raw u16 lanes, u16 lanes of w<<8}:
// every byte of the group appears once as the HIGH byte of a lane, so the group holds a byte
// outside [lo, hi]  <=>  some lane exceeds ((hi-lo)<<8 | 0xFF).
__device__ __forceinline__ uint32_t group_range_acc(const uint4& w, uint32_t negLB2) {
  uint32_t acc = __viaddmax_u16x2(w.x, negLB2, 0u);
  acc = __viaddmax_u16x2(w.x << 8, negLB2, acc);
  acc = __viaddmax_u16x2(w.y, negLB2, acc);
  acc = __viaddmax_u16x2(w.y << 8, negLB2, acc);
  acc = __viaddmax_u16x2(w.z, negLB2, acc);
  acc = __viaddmax_u16x2(w.z << 8, negLB2, acc);
  acc = __viaddmax_u16x2(w.w, negLB2, acc);
  acc = __viaddmax_u16x2(w.w << 8, negLB2, acc);
  return acc;
}

__global__ void __launch_bounds__(512, 1) td_u8_staged_kernel(const TdU8Params P) {
  extern __shared__ __align__(128) uint8_t smem[];
  const int lane = threadIdx.x & 31;
  const int warp = threadIdx.x >> 5;
  const int nwarps = blockDim.x >> 5;
  uint8_t* slot = smem + (size_t)warp * P.slot_bytes;
  uint16_t* queue = reinterpret_cast<uint16_t*>(smem + (size_t)nwarps * P.slot_bytes) + (size_t)warp * P.queue_entries;
  uint64_t* bar = reinterpret_cast<uint64_t*>(smem + (size_t)nwarps * P.slot_bytes +
                                              (size_t)nwarps * P.queue_entries * sizeof(uint16_t)) + warp;
  if (lane == 0) {
    mbar_init(bar, 1);
    fence_mbar_init();
  }
  __syncwarp();

  const int S = P.S;
  const uint32_t lt_mask = (1u << lane) - 1u;
  uint32_t phase = 0;
  const int64_t total_warps = (int64_t)gridDim.x * nwarps;
  for (int64_t row = (int64_t)blockIdx.x * nwarps + warp; row < P.rows; row += total_warps) {
    // ---------------------------------------------------------------- T1: load
    const uint8_t* g = P.src + row * P.stride;
    const int h = (int)(reinterpret_cast<uintptr_t>(g) & 15);   // row byte i lives at slot[h + i]
    int a0 = (16 - h) & 15;                                      // bytes before the first aligned address
    if (a0 > S) a0 = S;
    const int body = (S - a0) & ~15;                             // aligned interior, multiple of 16
    const int a1 = a0 + body;
    const int J = (h + S + 15) >> 4;                             // 16-byte groups covering the row
    if (lane == 0 && body > 0) {
      mbar_arrive_expect_tx(bar, (uint32_t)body);
      bulk_load(slot + h + a0, g + a0, (uint32_t)body, bar);
    }
    if (lane < 16) {
      if (lane < h) slot[lane] = 0;                              // padding in front of the row
      if (lane < a0) slot[h + lane] = g[lane];                   // head bytes
    } else {
      const int t = lane - 16;
      if (a1 + t < S) slot[h + a1 + t] = g[a1 + t];              // tail bytes
      if (h + S + t < 16 * J) slot[h + S + t] = 0;               // padding behind the row
    }
    if (body > 0) {
      mbar_wait(bar, phase);
      phase ^= 1;
    }
    __syncwarp();

    // ---------------------------------------------------------------- T2: statistics
    const uint4* s4 = reinterpret_cast<const uint4*>(slot);
    uint32_t s1 = 0, s2 = 0;
#pragma unroll 4
    for (int gi = lane; gi < J; gi += 32) {
      const uint4 w = s4[gi];
      s1 = __dp4a(w.x, 0x01010101u, s1); s2 = __dp4a(w.x, w.x, s2);
      s1 = __dp4a(w.y, 0x01010101u, s1); s2 = __dp4a(w.y, w.y, s2);
      s1 = __dp4a(w.z, 0x01010101u, s1); s2 = __dp4a(w.z, w.z, s2);
      s1 = __dp4a(w.w, 0x01010101u, s1); s2 = __dp4a(w.w, w.w, s2);
    }
    uint64_t Ssum = warp_sum_u32(s1);
    uint64_t Qsum = warp_sum_u64((uint64_t)s2);

    // ---------------------------------------------------------------- T3..T5: thresholds, on chip
    const int forced_first = (h > 0) ? 0 : -1;                   // groups holding padding are always revisited
    const int forced_last = ((h + S) & 15) ? J - 1 : -1;
    for (int it = 0; it < P.n_thr; ++it) {
      const U8Cut cut = make_cut_u8((uint32_t)S, Ssum, Qsum, P.p[it]);
      int lo, hi;
      warp_bounds_u8(cut, lane, lo, hi);
      if (lo == 0 && hi == 255) continue;                        // nothing can be cut
      const uint32_t r = rounded_mean_u8((uint32_t)S, Ssum);
      const bool all = lo > hi;
      const uint32_t neg = (0x10000u - ((uint32_t)lo << 8)) & 0xffffu;
      const uint32_t negLB2 = neg | (neg << 16);
      const uint32_t thr = (((uint32_t)(hi - lo) << 8) | 0xffu) & 0xffffu;
      const uint32_t thr2 = thr | (thr << 16);
      // T4a: packed range check, queue the groups that hold a value outside [lo, hi]
      int qn = 0;
#pragma unroll 2
      for (int g0 = 0; g0 < J; g0 += 32) {
        const int gi = g0 + lane;
        bool hit = false;
        if (gi < J) {
          const uint32_t acc = group_range_acc(s4[gi], negLB2);
          hit = all || (__vmaxu2(acc, thr2) != thr2) || gi == forced_first || gi == forced_last;
        }
        const uint32_t b = __ballot_sync(FULL, hit);
        if (b) {
          if (hit) queue[qn + __popc(b & lt_mask)] = (uint16_t)gi;
          qn += __popc(b);
        }
      }
      __syncwarp();
      // T4b: revisit the queued groups byte by byte (two groups per warp step)
      uint32_t cnt = 0, sx = 0, sxx = 0;
      for (int e = lane >> 4; e < qn; e += 2) {
        const int pos = (int)queue[e] * 16 + (lane & 15);
        const int i = pos - h;
        if ((unsigned)i < (unsigned)S) {
          const uint32_t x = slot[pos];
          if ((int)x < lo || (int)x > hi) {
            slot[pos] = (uint8_t)r;
            ++cnt; sx += x; sxx += x * x;
            if (P.flags) P.flags[row * S + i] = 1;
          }
        }
      }
      cnt = warp_sum_u32(cnt);
      if (cnt) {
        sx = warp_sum_u32(sx);
        const uint64_t sxx64 = warp_sum_u64((uint64_t)sxx);
        Ssum = Ssum + (uint64_t)cnt * r - sx;
        Qsum = Qsum + (uint64_t)cnt * r * r - sxx64;
        if (lane == 0 && P.counts) atomicAdd(&P.counts[it], (unsigned long long)cnt);
      }
      __syncwarp();
    }

    // ---------------------------------------------------------------- T6: store
    uint8_t* go = P.dst + row * P.stride;
    fence_proxy_async_smem();
    __syncwarp();
    if (lane == 0 && body > 0) {
      bulk_store(go + a0, slot + h + a0, (uint32_t)body);
      bulk_commit();
    }
    if (lane < 16) {
      if (lane < a0) go[lane] = slot[h + lane];
    } else {
      const int t = lane - 16;
      if (a1 + t < S) go[a1 + t] = slot[h + a1 + t];
    }
    if (lane == 0 && body > 0) bulk_wait_read<0>();               // slot may be overwritten after this
    __syncwarp();
  }
}

// ------------------------------------------------------------------------------------------------
// generic path
// ------------------------------------------------------------------------------------------------
constexpr int kGenericThreads = 256;

__device__ __forceinline__ uint64_t block_sum_u64(uint64_t v, uint64_t* red) {
  v = warp_sum_u64(v);
  __syncthreads();
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
  __syncthreads();
  uint64_t t = 0;
  for (int w = 0; w < (int)(blockDim.x >> 5); ++w) t += red[w];
  return t;
}

// lower median (rank (n-1)/2) from a 256-bin histogram, computed by warp 0; result to *out
__device__ __forceinline__ void warp_hist_median(const uint32_t* hist, uint32_t n, int lane, int* out) {
  uint32_t c[8], tot = 0;
#pragma unroll
  for (int j = 0; j < 8; ++j) { c[j] = hist[lane * 8 + j]; tot += c[j]; }
  uint32_t incl = tot;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const uint32_t t = __shfl_up_sync(FULL, incl, o);
    if (lane >= o) incl += t;
  }
  const uint32_t rank = (n - 1) / 2;
  uint32_t before = incl - tot;                                   // values in lower lanes
  if (rank >= before && rank < incl) {
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      if (rank < before + c[j]) { *out = lane * 8 + j; break; }
      before += c[j];
    }
  }
}

__global__ void __launch_bounds__(kGenericThreads) td_u8_generic_kernel(const TdU8Params P) {
  __shared__ uint64_t red[kGenericThreads / 32];
  __shared__ uint32_t hist[256];
  __shared__ int sh_lo, sh_hi, sh_r;
  const int tid = threadIdx.x, lane = tid & 31;
  for (int64_t row = blockIdx.x; row < P.rows; row += gridDim.x) {
    const uint8_t* s = P.src + row * P.stride;
    uint8_t* d = P.dst + row * P.stride;
    for (int w0 = 0; w0 < P.S; w0 += P.window) {
      const int n = min(P.window, P.S - w0);
      uint64_t a = 0, b = 0;
      for (int i = tid; i < n; i += kGenericThreads) {
        const uint32_t x = s[w0 + i];
        if (d != s) d[w0 + i] = (uint8_t)x;
        a += x; b += x * x;
      }
      uint64_t Ssum = block_sum_u64(a, red);
      uint64_t Qsum = block_sum_u64(b, red);
      for (int it = 0; it < P.n_thr; ++it) {
        if (P.policy == 1) {                                      // lower median of the snapshot
          for (int i = tid; i < 256; i += kGenericThreads) hist[i] = 0;
          __syncthreads();
          for (int i = tid; i < n; i += kGenericThreads) atomicAdd(&hist[d[w0 + i]], 1u);
          __syncthreads();
        }
        if (tid < 32) {
          const U8Cut cut = make_cut_u8((uint32_t)n, Ssum, Qsum, P.p[it]);
          int lo, hi;
          warp_bounds_u8(cut, lane, lo, hi);
          if (lane == 0) { sh_lo = lo; sh_hi = hi; }
          if (P.policy == 1) warp_hist_median(hist, (uint32_t)n, lane, &sh_r);
          else if (lane == 0) sh_r = (int)rounded_mean_u8((uint32_t)n, Ssum);
        }
        __syncthreads();
        const int lo = sh_lo, hi = sh_hi;
        const uint32_t r = (uint32_t)sh_r;
        uint64_t cnt = 0, sx = 0, sxx = 0;
        if (!(lo == 0 && hi == 255)) {
          for (int i = tid; i < n; i += kGenericThreads) {
            const uint32_t x = d[w0 + i];
            if ((int)x < lo || (int)x > hi) {
              d[w0 + i] = (uint8_t)r;
              ++cnt; sx += x; sxx += x * x;
              if (P.flags) P.flags[row * P.S + w0 + i] = 1;
            }
          }
        }
        cnt = block_sum_u64(cnt, red);
        sx = block_sum_u64(sx, red);
        sxx = block_sum_u64(sxx, red);
        Ssum = Ssum + cnt * r - sx;
        Qsum = Qsum + cnt * r * r - sxx;
        if (tid == 0 && P.counts && cnt) atomicAdd(&P.counts[it], (unsigned long long)cnt);
        __syncthreads();
      }
    }
  }
}

}  // namespace rfim
