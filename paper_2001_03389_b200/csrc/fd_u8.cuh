// fd_u8.cuh -- frequency-domain sigma cut (FDSC, Fig. 3) for uint8 dynamic spectra,
// one bin of all channels (BASELINE.json configs[2]).
//
// Two kernels:
//   fd_u8_tile_kernel   the hot path.  A CTA owns a tile of all C channels x Ts consecutive samples of
//       one beam.  F1: the tile is brought into shared memory by TMA tensor copies issued by one thread.
//       Rows of a dense [C][S] beam are only 4-byte aligned (12500 mod 16 = 4) while a tensor map needs
//       16-byte strides AND 16-byte aligned box starts (measured: a box whose inner coordinate is not a
//       multiple of 16 bytes faults).  So the rows are split into m = 16/gcd(pitch,16) alignment classes
//       (row mod m): class r is a 2-D tensor with row stride m*pitch whose base is rounded DOWN to 16
//       bytes (by off_r bytes), and every box is 16 bytes wider than the tile (kExact = false): the
//       wanted samples sit off_r bytes into each shared-memory row.  When every row is 16-byte aligned
//       (padded pitch; kExact = true) the boxes are exact and the tile is also stored by TMA.
//       F2: a thread owns one 32-bit word column (4 samples) and every 16th row; 4x4 byte transposes
//       (PRMT) turn four rows into four words that each hold ONE column, so that IDP.4A gives the exact
//       column sums and sums of squares.  F3: one thread per column evaluates the exact integer
//       predicate around a float estimate -> [lo, hi], r.  F4: packed range check with per-column bounds
//       (VIADDMNMX.U16x2, 3 instructions per word, eight rows per test); only groups with a hit are
//       revisited byte by byte (replace in shared memory, update the column's S, Q, count with
//       shared-memory atomics).  F5: next threshold, on chip.  F6: TMA tensor stores (kExact) or
//       coalesced 32-bit stores of exactly the tile's bytes.  HBM sees one read and one write per sample.
//   fd_u8_generic_kernel  any pitch / alignment / channel count: one thread per (beam, sample) column,
//       iterations through global memory (L2).  Correctness path, not tuned.
#pragma once

#include <cuda.h>   // CUtensorMap (types only: the encoder is fetched through the runtime, no -lcuda)

#include "common.cuh"

namespace rfim {

constexpr int kFdMaxClasses = 4;

struct FdMaps {
  CUtensorMap src[kFdMaxClasses];
  CUtensorMap dst[kFdMaxClasses];
};

struct FdU8Params {
  const uint8_t* src;
  uint8_t* dst;
  int64_t stride;
  int beams, C, S;
  int n_thr;
  uint32_t p[16];
  float pf[16];
  uint8_t* flags;               // optional [beams][C][S]
  unsigned long long* counts;   // optional [n_thr]
  // tile kernel
  int m;                        // alignment classes
  int rows_per_class;           // C / m
  int box_rows;                 // rows per TMA box (divides rows_per_class, <= 256)
  int off[kFdMaxClasses];       // x offset (bytes) of class r inside its 16-byte aligned tensor
  int tiles_per_beam;
  int64_t total_tiles;
};

// ---------------------------------------------------------------- TMA tensor copies (2-D, tiled)
__device__ __forceinline__ void tma_load_2d(void* smem_dst, const CUtensorMap* map, int x, int y, uint64_t* bar) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
      ::"r"(smem_addr(smem_dst)), "l"(reinterpret_cast<uint64_t>(map)), "r"(x), "r"(y), "r"(smem_addr(bar))
      : "memory");
}
__device__ __forceinline__ void tma_store_2d(const CUtensorMap* map, int x, int y, const void* smem_src) {
  asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.tile.bulk_group [%0, {%1, %2}], [%3];" ::"l"(
                   reinterpret_cast<uint64_t>(map)),
               "r"(x), "r"(y), "r"(smem_addr(smem_src))
               : "memory");
}
__device__ __forceinline__ void tma_prefetch_desc(const CUtensorMap* map) {
  asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(map)) : "memory");
}

__device__ __forceinline__ uint32_t prmt_b32(uint32_t a, uint32_t b, uint32_t sel) {
  uint32_t d;
  asm("prmt.b32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(sel));
  return d;
}

// Kept interval for one cut, ONE thread: float estimate of mu -/+ k sigma, then a short walk on the
// EXACT predicate to the true ends (the kept set is an interval).  Falls back to the bisection of
// thread_bounds_u8 when the estimate is not next to a kept value.  Result identical to warp_bounds_u8.
__device__ __forceinline__ void thread_bounds_u8_fast(const U8Cut& c, float k, uint64_t V, int& lo, int& hi) {
  const float rn = __frcp_rn((float)c.N);
  const float mu = (float)c.S * rn;
  const float vf = (float)V;
  const float ks = k * (vf * rsqrtf(fmaxf(vf, 1.0f))) * rn;
  int x = (int)fminf(fmaxf(ceilf(mu - ks), 0.0f), 255.0f);
  int y = (int)fminf(fmaxf(floorf(mu + ks), 0.0f), 255.0f);
  int steps = 0;
  while (cut_flags_u8(c, (uint32_t)x) && steps < 3 && x < 255) { ++x; ++steps; }
  steps = 0;
  while (cut_flags_u8(c, (uint32_t)y) && steps < 3 && y > 0) { --y; ++steps; }
  if (cut_flags_u8(c, (uint32_t)x) || cut_flags_u8(c, (uint32_t)y) || x > y) {
    thread_bounds_u8(c, lo, hi);
    return;
  }
  while (x > 0 && !cut_flags_u8(c, (uint32_t)(x - 1))) --x;
  while (y < 255 && !cut_flags_u8(c, (uint32_t)(y + 1))) ++y;
  lo = x;
  hi = y;
}

// Exact 0xFF-per-byte mask of the bytes of w outside their column's [lo, hi]; constants per u16 lane:
// chiE/cloE for bytes 0 and 2, chiO/cloO for bytes 1 and 3 (see bytes_outside in td_u8.cuh).
__device__ __forceinline__ uint32_t bytes_outside_cols(uint32_t w, uint32_t chiE, uint32_t cloE, uint32_t chiO,
                                                       uint32_t cloO) {
  const uint32_t xe = prmt_b32(w, 0u, 0x4240u), xo = prmt_b32(w, 0u, 0x4341u);
  const uint32_t fe = (xe + chiE) | ~(xe + cloE);
  const uint32_t fo = (xo + chiO) | ~(xo + cloO);
  return prmt_b32(fe, fo, 0xFBD9u);
}

// shared-memory control block behind the tile
constexpr int kFdRG = 16;                    // row groups: a thread owns every 16th row of each class
template <int Ts>
struct FdSmem {
  static constexpr int WC = Ts / 4;          // word columns
  uint64_t bar;
  uint32_t red[kFdRG * WC * 8];              // per row group, per word column: S[4], Q[4]
  uint32_t dS[Ts], dQ[Ts], dcnt[Ts];         // per column updates of one iteration (atomics)
  uint32_t lo4[WC], hi4[WC], r4[WC];         // per word column: packed bounds and replacement values
  uint32_t any_cut;                          // some column of the tile has bounds inside 0..255
};

// Ts samples per tile; 4*Ts threads (Ts/4 word columns x 16 row groups).  kExact: rows are 16-byte
// aligned, boxes are exactly Ts wide and the tile is stored by TMA; else boxes are Ts+16 wide.
template <int Ts, bool kExact>
__global__ void __launch_bounds__(4 * Ts) fd_u8_tile_kernel(const __grid_constant__ FdMaps maps, const FdU8Params P) {
  using Sm = FdSmem<Ts>;
  constexpr int WC = Sm::WC, RG = kFdRG, NT = 4 * Ts;
  constexpr int PW = kExact ? WC : WC + 4;                                // shared-memory row pitch in words
  extern __shared__ __align__(128) uint8_t smem[];
  const int C = P.C, Rc = P.rows_per_class;
  uint32_t* tile = reinterpret_cast<uint32_t*>(smem);                     // [C][PW] words, class-major rows
  Sm& sm = *reinterpret_cast<Sm*>(smem + (((size_t)C * PW * 4 + 127) & ~(size_t)127));
  const int tid = threadIdx.x;
  const int wc = tid % WC, rg = tid / WC;
  const int nk = (Rc - rg + RG - 1) / RG;             // rows rg, rg+RG, ... of this thread inside EACH class
  // word offset of the tile's first sample inside a shared-memory row of class r
  auto wofs = [&](int r) { return kExact ? 0 : (P.off[r] >> 2); };

  if (tid == 0) {
    mbar_init(&sm.bar, 1);
    fence_mbar_init();
    for (int r = 0; r < P.m; ++r) { tma_prefetch_desc(&maps.src[r]); if (kExact) tma_prefetch_desc(&maps.dst[r]); }
  }
  for (int i = tid; i < Ts; i += NT) { sm.dS[i] = 0; sm.dQ[i] = 0; sm.dcnt[i] = 0; }
  __syncthreads();

  uint32_t phase = 0;
  const int nbox = Rc / P.box_rows;
  for (int64_t t = blockIdx.x; t < P.total_tiles; t += gridDim.x) {
    const int b = (int)(t / P.tiles_per_beam);
    const int s0 = (int)(t % P.tiles_per_beam) * Ts;
    // ------------------------------------------------------------------ F1: load the tile
    if (tid == 0) {
      mbar_arrive_expect_tx(&sm.bar, (uint32_t)(C * PW * 4));
      for (int r = 0; r < P.m; ++r)
        for (int bx = 0; bx < nbox; ++bx) {
          const int row0 = r * Rc + bx * P.box_rows;
          // kExact: off[r] == 0.  Otherwise x = s0 addresses byte s0 - off[r] of the row (never before the
          // row's 16-byte aligned tensor origin) and the box is 16 bytes wider than the tile.
          tma_load_2d(tile + (size_t)row0 * PW, &maps.src[r], s0, b * Rc + bx * P.box_rows, &sm.bar);
        }
    }
    mbar_wait(&sm.bar, phase);
    phase ^= 1;

    // ------------------------------------------------------------------ F2: column statistics
    uint32_t S4[4] = {0, 0, 0, 0}, Q4[4] = {0, 0, 0, 0};
    for (int cls = 0; cls < P.m; ++cls) {
      const uint32_t* col = tile + (size_t)(cls * Rc + rg) * PW + wofs(cls) + wc;
      int k = 0;
#pragma unroll 2
      for (; k + 4 <= nk; k += 4) {
        const uint32_t a = col[(size_t)(k + 0) * RG * PW], bb = col[(size_t)(k + 1) * RG * PW];
        const uint32_t c = col[(size_t)(k + 2) * RG * PW], d = col[(size_t)(k + 3) * RG * PW];
        const uint32_t ab_lo = prmt_b32(a, bb, 0x5140u), ab_hi = prmt_b32(a, bb, 0x7362u);
        const uint32_t cd_lo = prmt_b32(c, d, 0x5140u), cd_hi = prmt_b32(c, d, 0x7362u);
        const uint32_t t0 = prmt_b32(ab_lo, cd_lo, 0x5410u), t1 = prmt_b32(ab_lo, cd_lo, 0x7632u);
        const uint32_t t2 = prmt_b32(ab_hi, cd_hi, 0x5410u), t3 = prmt_b32(ab_hi, cd_hi, 0x7632u);
        S4[0] = __dp4a(t0, 0x01010101u, S4[0]); Q4[0] = __dp4a(t0, t0, Q4[0]);
        S4[1] = __dp4a(t1, 0x01010101u, S4[1]); Q4[1] = __dp4a(t1, t1, Q4[1]);
        S4[2] = __dp4a(t2, 0x01010101u, S4[2]); Q4[2] = __dp4a(t2, t2, Q4[2]);
        S4[3] = __dp4a(t3, 0x01010101u, S4[3]); Q4[3] = __dp4a(t3, t3, Q4[3]);
      }
      for (; k < nk; ++k) {
        const uint32_t w = col[(size_t)k * RG * PW];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          const uint32_t x = (w >> (8 * j)) & 0xffu;
          S4[j] += x; Q4[j] += x * x;
        }
      }
    }
    {
      uint32_t* r = sm.red + (size_t)(rg * WC + wc) * 8;
#pragma unroll
      for (int j = 0; j < 4; ++j) { r[j] = S4[j]; r[4 + j] = Q4[j]; }
    }
    __syncthreads();
    // thread t < Ts owns column t: its S and Q live in registers across the iterations
    uint32_t colS = 0, colQ = 0;
    if (tid < Ts) {
      const int cw = tid >> 2, cj = tid & 3;
#pragma unroll
      for (int g = 0; g < RG; ++g) {
        colS += sm.red[(size_t)(g * WC + cw) * 8 + cj];
        colQ += sm.red[(size_t)(g * WC + cw) * 8 + 4 + cj];
      }
    }

    // ------------------------------------------------------------------ F3..F5: thresholds, on chip
    for (int it = 0; it < P.n_thr; ++it) {
      if (tid == 0) sm.any_cut = 0;
      __syncthreads();
      if (tid < Ts) {
        int lo, hi;
        const uint64_t V = (uint64_t)C * colQ - (uint64_t)colS * colS;
        const U8Cut cut = make_cut_u8((uint32_t)C, colS, V, P.p[it]);
        thread_bounds_u8_fast(cut, P.pf[it], V, lo, hi);
        // Columns past the end of the row (last tile) are inert.  TMA checks the inner bound in 16-byte
        // units (measured), so they may hold the next row's first bytes rather than zeros.
        if (s0 + tid >= P.S) { lo = 0; hi = 255; }
        const uint32_t r = rounded_mean_u8((uint32_t)C, colS);
        reinterpret_cast<uint8_t*>(sm.lo4)[tid] = (uint8_t)lo;
        reinterpret_cast<uint8_t*>(sm.hi4)[tid] = (uint8_t)hi;
        reinterpret_cast<uint8_t*>(sm.r4)[tid] = (uint8_t)r;
        if (!(lo == 0 && hi == 255)) sm.any_cut = 1;
      }
      __syncthreads();
      if (sm.any_cut == 0) continue;                               // uniform: nothing can be cut in this tile
      // F4a: packed range check, per-column bounds in the u16 lanes
      const uint32_t lo4 = sm.lo4[wc], hi4 = sm.hi4[wc], r4 = sm.r4[wc];
      uint32_t lob[4], hib[4];
#pragma unroll
      for (int j = 0; j < 4; ++j) { lob[j] = (lo4 >> (8 * j)) & 0xffu; hib[j] = (hi4 >> (8 * j)) & 0xffu; }
      // odd chain: bytes 1 and 3 are the high bytes of the u16 lanes of w; even chain: bytes 0, 2 of w << 8
      auto neg16 = [](uint32_t lo) { return (0x10000u - (lo << 8)) & 0xffffu; };
      auto thr16 = [](uint32_t lo, uint32_t hi) { return lo > hi ? 0u : (((hi - lo) << 8) | 0xffu); };
      auto ini16 = [](uint32_t lo, uint32_t hi) { return lo > hi ? 1u : 0u; };   // empty interval: always a hit
      const uint32_t negO = neg16(lob[1]) | (neg16(lob[3]) << 16), negE = neg16(lob[0]) | (neg16(lob[2]) << 16);
      const uint32_t thrO = thr16(lob[1], hib[1]) | (thr16(lob[3], hib[3]) << 16);
      const uint32_t thrE = thr16(lob[0], hib[0]) | (thr16(lob[2], hib[2]) << 16);
      const uint32_t iniO = ini16(lob[1], hib[1]) | (ini16(lob[3], hib[3]) << 16);
      const uint32_t iniE = ini16(lob[0], hib[0]) | (ini16(lob[2], hib[2]) << 16);
      const uint32_t chiE = (0x7fffu - hib[0]) | ((0x7fffu - hib[2]) << 16), cloE = (0x8000u - lob[0]) | ((0x8000u - lob[2]) << 16);
      const uint32_t chiO = (0x7fffu - hib[1]) | ((0x7fffu - hib[3]) << 16), cloO = (0x8000u - lob[1]) | ((0x8000u - lob[3]) << 16);
      const bool last = (it == P.n_thr - 1);
      const bool need_stats = !last;
      const bool need_cnt = P.counts != nullptr;

      for (int cls = 0; cls < P.m; ++cls) {
        uint32_t* col = tile + (size_t)(cls * Rc + rg) * PW + wofs(cls) + wc;
        // F4b: exact fix of one word (rare path)
        auto fix_word = [&](int k, uint32_t w) {
          const uint32_t msk = bytes_outside_cols(w, chiE, cloE, chiO, cloO);
          if (msk == 0) return;
          col[(size_t)k * RG * PW] = (w & ~msk) | (r4 & msk);
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            if ((msk >> (8 * j)) & 1u) {
              const uint32_t x = (w >> (8 * j)) & 0xffu, r = (r4 >> (8 * j)) & 0xffu;
              const int colj = wc * 4 + j;
              if (need_stats) {
                atomicAdd(&sm.dS[colj], r - x);
                atomicAdd(&sm.dQ[colj], r * r - x * x);
              }
              if (need_cnt) atomicAdd(&sm.dcnt[colj], 1u);
              if (P.flags) {
                const int ch = (rg + k * RG) * P.m + cls;          // row g of class cls is channel g*m + cls
                P.flags[((int64_t)b * C + ch) * P.S + s0 + colj] = 1;
              }
            }
          }
        };
        int k = 0;
        for (; k + 8 <= nk; k += 8) {
          uint32_t w[8];
#pragma unroll
          for (int u = 0; u < 8; ++u) w[u] = col[(size_t)(k + u) * RG * PW];
          uint32_t accO = iniO, accE = iniE;
#pragma unroll
          for (int u = 0; u < 8; ++u) {
            accO = __viaddmax_u16x2(w[u], negO, accO);
            accE = __viaddmax_u16x2(w[u] << 8, negE, accE);
          }
          if (__vmaxu2(accO, thrO) != thrO || __vmaxu2(accE, thrE) != thrE) {
#pragma unroll
            for (int u = 0; u < 8; ++u) fix_word(k + u, w[u]);
          }
        }
        for (; k < nk; ++k) fix_word(k, col[(size_t)k * RG * PW]);
      }
      __syncthreads();
      if (tid < Ts && (need_stats || need_cnt)) {
        if (need_stats) {
          colS += sm.dS[tid];
          colQ += sm.dQ[tid];
          sm.dS[tid] = 0;
          sm.dQ[tid] = 0;
        }
        if (need_cnt) {
          const uint32_t cnt = sm.dcnt[tid];
          sm.dcnt[tid] = 0;
          if (cnt) atomicAdd(&P.counts[it], (unsigned long long)cnt);
        }
      }
    }

    // ------------------------------------------------------------------ F6: store the tile
    if (kExact && s0 + Ts <= P.S) {                                 // (a ragged last tile is stored by the lanes:
      fence_proxy_async_smem();                                     //  TMA stores clip in 16-byte units, measured)
      __syncthreads();
      if (tid == 0) {
        for (int r = 0; r < P.m; ++r)
          for (int bx = 0; bx < nbox; ++bx) {
            const int row0 = r * Rc + bx * P.box_rows;
            tma_store_2d(&maps.dst[r], s0, b * Rc + bx * P.box_rows, tile + (size_t)row0 * PW);
          }
        bulk_commit();
        bulk_wait_read<0>();                                        // the tile may be overwritten after this
      }
      __syncthreads();
    } else {
      __syncthreads();
      const int s = s0 + wc * 4;                                    // first sample of this thread's word column
      if (s < P.S) {
        const bool whole = s + 4 <= P.S;
        for (int cls = 0; cls < P.m; ++cls) {
          const uint32_t* col = tile + (size_t)(cls * Rc + rg) * PW + wofs(cls) + wc;
          uint8_t* g = P.dst + ((int64_t)b * C + (int64_t)rg * P.m + cls) * P.stride + s;
          const int64_t gstep = (int64_t)RG * P.m * P.stride;
          if (whole) {
#pragma unroll 4
            for (int k = 0; k < nk; ++k) *reinterpret_cast<uint32_t*>(g + k * gstep) = col[(size_t)k * RG * PW];
          } else {
            for (int k = 0; k < nk; ++k) {
              const uint32_t w = col[(size_t)k * RG * PW];
              for (int j = 0; s + j < P.S; ++j) g[k * gstep + j] = (uint8_t)(w >> (8 * j));
            }
          }
        }
      }
      __syncthreads();                                              // the tile may be overwritten after this
    }
  }
  if (kExact && tid == 0) bulk_wait_all<0>();
}

// ------------------------------------------------------------------------------------------------
// generic path: one thread per (beam, sample) column
// ------------------------------------------------------------------------------------------------
constexpr int kFdGenericThreads = 128;

__global__ void __launch_bounds__(kFdGenericThreads) fd_u8_generic_kernel(const FdU8Params P) {
  const int64_t ncol = (int64_t)P.beams * P.S;
  for (int64_t col = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; col < ncol;
       col += (int64_t)gridDim.x * blockDim.x) {
    const int b = (int)(col / P.S), s = (int)(col % P.S);
    const uint8_t* src = P.src + (int64_t)b * P.C * P.stride + s;
    uint8_t* dst = P.dst + (int64_t)b * P.C * P.stride + s;
    uint32_t S = 0;
    uint64_t Q = 0;
    for (int c = 0; c < P.C; ++c) {
      const uint32_t x = src[(int64_t)c * P.stride];
      if (dst != src) dst[(int64_t)c * P.stride] = (uint8_t)x;
      S += x; Q += x * x;
    }
    for (int it = 0; it < P.n_thr; ++it) {
      const uint64_t V = (uint64_t)P.C * Q - (uint64_t)S * S;
      const U8Cut cut = make_cut_u8((uint32_t)P.C, S, V, P.p[it]);
      int lo, hi;
      thread_bounds_u8(cut, lo, hi);
      if (lo == 0 && hi == 255) continue;
      const uint32_t r = rounded_mean_u8((uint32_t)P.C, S);
      uint32_t cnt = 0;
      for (int c = 0; c < P.C; ++c) {
        const uint32_t x = dst[(int64_t)c * P.stride];
        if ((int)x < lo || (int)x > hi) {
          dst[(int64_t)c * P.stride] = (uint8_t)r;
          ++cnt;
          S += r - x;
          Q += (uint64_t)(r * r) - (uint64_t)(x * x);
          if (P.flags) P.flags[((int64_t)b * P.C + c) * P.S + s] = 1;
        }
      }
      if (cnt && P.counts) atomicAdd(&P.counts[it], (unsigned long long)cnt);
    }
  }
}

}  // namespace rfim
