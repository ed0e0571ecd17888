// fd_u8.cuh -- frequency-domain sigma cut (FDSC, Fig. 3) for uint8 dynamic spectra,
// one bin of all channels (BASELINE.json configs[2]).
//
// Two kernels:
//   fd_u8_cluster_kernel   the hot path.  A thread-block CLUSTER of CL CTAs owns a tile of all C
//       channels x Ts consecutive samples of one beam; CTA q of the cluster holds channels
//       [q*Rq, (q+1)*Rq) of the tile in its shared memory.  Splitting the channels over a cluster is
//       what lets the row segments be long (Ts ~ 500 bytes for C = 1536, CL = 8): FDSC wants whole
//       columns on chip while HBM wants long contiguous rows.
//       F1: every row segment is one 1-D TMA bulk copy (cp.async.bulk) of the 16-byte aligned
//       superset of its bytes, issued by one thread per row, all completing on one mbarrier.  Rows of
//       a dense [C][S] beam are only 4-byte aligned (12500 mod 16 = 4), so row r lands off_r =
//       (address mod 16) bytes into its shared-memory row; off_r is constant for the rows one thread
//       owns (they are 4 apart and 4 * pitch is a multiple of 16).
//       F2: a thread owns one 32-bit word column (4 samples) and every 4th row of the CTA; 4x4 byte
//       transposes (PRMT) turn four rows into four words that each hold ONE column, so IDP.4A gives
//       exact column sums and sums of squares.  Partial sums are reduced over the four row groups by
//       shuffles and over the cluster through distributed shared memory (DSMEM).
//       F3: column c is owned by one thread of one CTA of the cluster, which keeps (S, Q) in
//       registers over the iterations, evaluates the exact integer predicate around a float estimate
//       -> [lo, hi], r, and publishes them (with packed range-check constants); the other CTAs pull
//       them through DSMEM.
//       F4: packed range check with per-column bounds (VIADDMNMX.U16x2, 3 instructions per word);
//       only words with a hit are revisited with exact byte masks (replace in shared memory,
//       accumulate the column deltas in packed registers).  F5: next threshold, on chip.
//       F6: every row segment is stored by one bulk copy of its 16-byte aligned interior plus a few
//       32-bit / byte stores for the ragged ends.  HBM sees one read and one write per sample.
//   fd_u8_generic_kernel  any pitch / alignment / channel count: one thread per (beam, sample) column,
//       iterations through global memory (L2).  Correctness path, not tuned.
#pragma once

#include "common.cuh"

namespace rfim {

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
  // cluster kernel
  int Ts;                       // tile width in samples (multiple of 4, <= 4*PW - 16)
  int WC;                       // word columns per tile, rounded up to a multiple of 8; blockDim = 4*WC
  int Rq;                       // channels per CTA = ceil(C / cluster size)
  int tiles_per_beam;
  int64_t total_tiles;
};

__device__ __forceinline__ uint32_t prmt_b32(uint32_t a, uint32_t b, uint32_t sel) {
  uint32_t d;
  asm("prmt.b32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(sel));
  return d;
}

// ---------------------------------------------------------------- cluster helpers
__device__ __forceinline__ uint32_t cluster_ctarank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
  return r;
}
__device__ __forceinline__ uint32_t cluster_nctarank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_nctarank;" : "=r"(r));
  return r;
}
__device__ __forceinline__ uint32_t cluster_id_x() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%clusterid.x;" : "=r"(r));
  return r;
}
__device__ __forceinline__ uint32_t cluster_nid_x() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%nclusterid.x;" : "=r"(r));
  return r;
}
// barrier over all threads of all CTAs of the cluster; orders shared-memory accesses cluster-wide
__device__ __forceinline__ void cluster_sync_all() {
  asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// address of the same shared-memory location in CTA `rank` of the cluster
__device__ __forceinline__ uint32_t dsmem_addr(const void* local, uint32_t rank) {
  uint32_t ra;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(ra) : "r"(smem_addr(local)), "r"(rank));
  return ra;
}
__device__ __forceinline__ uint32_t dsmem_ld_u32(uint32_t addr) {
  uint32_t v;
  asm volatile("ld.shared::cluster.u32 %0, [%1];" : "=r"(v) : "r"(addr));
  return v;
}
__device__ __forceinline__ uint4 dsmem_ld_u128(uint32_t addr) {
  uint4 v;
  asm volatile("ld.shared::cluster.v4.u32 {%0, %1, %2, %3}, [%4];"
               : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w)
               : "r"(addr)
               : "memory");
  return v;
}

// colS += sum over the cluster of *pS, colQ += sum of *pQ.  All (up to 16) remote loads are issued before the
// first is consumed: a DSMEM load takes about 200 cycles, a loop of dependent adds would pay that per CTA.
__device__ __forceinline__ void cluster_gather2(const uint32_t* pS, const uint32_t* pQ, uint32_t ncta, uint32_t& colS,
                                                uint32_t& colQ) {
  uint32_t vs[8], vq[8];
#pragma unroll
  for (uint32_t q = 0; q < 8; ++q) {
    vs[q] = 0; vq[q] = 0;
    if (q < ncta) {
      vs[q] = dsmem_ld_u32(dsmem_addr(pS, q));
      vq[q] = dsmem_ld_u32(dsmem_addr(pQ, q));
    }
  }
#pragma unroll
  for (uint32_t q = 0; q < 8; ++q) { colS += vs[q]; colQ += vq[q]; }
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

// ---------------------------------------------------------------- cluster kernel
// Shared memory of one CTA (PW = row pitch in 32-bit words, PW mod 32 in {8, 24} so that the four row
// groups of a warp fall into disjoint banks; TsP = 4 * WC padded columns):
//   tile  [Rq][PW] words      the CTA's channels of the tile
//   xS, xQ [TsP] u32          exchange: this CTA's partial column sums, later its column deltas
//   chk   [WC] uint4          per word column {negE, negO, thrE, thrO}: packed range-check constants
//   lo, hi, rr [TsP] bytes    per column kept interval and replacement (exact fix path)
//   bar, misc
constexpr int kFdRG = 4;   // row groups: a thread owns rows rg, rg + 4, ... of its CTA

__host__ __device__ inline size_t fd_cluster_ctrl_bytes(int WC) { return (size_t)WC * 4 * 15 + 64; }
__host__ __device__ inline size_t fd_cluster_smem_bytes(int PW, int Rq, int WC) {
  return (size_t)Rq * PW * 4 + fd_cluster_ctrl_bytes(WC);
}

// RG = row groups that share a warp: RG = 4 maps a warp to 8 word columns x 4 row groups (512 threads for a
// 128-word tile, each thread sees every 4th row of the CTA); RG = 1 maps a thread to one word column and
// ALL rows of the CTA (128 threads): four times the work per thread, so the per-tile overhead (bounds,
// exchanges, barriers, copies) is amortised over four times as many words, and no shuffles are needed.
template <int PW, int RG>
__global__ void __launch_bounds__(128 * RG, 2) fd_u8_cluster_kernel(const FdU8Params P) {
  extern __shared__ __align__(128) uint8_t smem[];
  const int C = P.C, Ts = P.Ts, WC = P.WC, Rq = P.Rq, TsP = 4 * WC;
  uint32_t* tile = reinterpret_cast<uint32_t*>(smem);
  uint8_t* ctrl = smem + (size_t)Rq * PW * 4;
  uint32_t* xS = reinterpret_cast<uint32_t*>(ctrl);
  uint32_t* xQ = xS + TsP;
  uint4* chk = reinterpret_cast<uint4*>(xQ + TsP);
  uint8_t* lo_b = reinterpret_cast<uint8_t*>(chk + WC);
  uint8_t* hi_b = lo_b + TsP;
  uint8_t* rr_b = hi_b + TsP;
  uint64_t* bar = reinterpret_cast<uint64_t*>(rr_b + TsP);
  volatile uint32_t* any_empty = reinterpret_cast<volatile uint32_t*>(bar + 1);

  const int tid = threadIdx.x, nthreads = blockDim.x, lane = tid & 31;
  const int j = RG == 4 ? (tid >> 5) * 8 + (lane & 7) : tid;   // word column of this thread
  const int rg0 = RG == 4 ? lane >> 3 : 0;            // first row group of this thread (it owns rg0, rg0 + RG, .. < 4)
  const uint32_t rank = cluster_ctarank(), ncta = cluster_nctarank();
  const int c0 = (int)rank * Rq;                      // first channel of this CTA
  const int nrows = max(0, min(Rq, C - c0));
  const int wpc = (WC + (int)ncta - 1) / (int)ncta;   // word columns owned per CTA (F3)
  const int nload = min(nrows, nthreads);

  if (tid == 0) {
    mbar_init(bar, nload > 0 ? nload : 1);
    fence_mbar_init();
    *any_empty = 0;
  }
  __syncthreads();
  if (ncta > 1) cluster_sync_all();                   // peers' shared memory is live before any DSMEM access

  uint32_t phase = 0;
  const uint32_t nclusters = cluster_nid_x();
  for (int64_t t = cluster_id_x(); t < P.total_tiles; t += nclusters) {
    const int b = (int)(t / P.tiles_per_beam);
    const int s0 = (int)(t % P.tiles_per_beam) * Ts;
    const int tw = min(Ts, P.S - s0);                 // valid columns of this tile
    const uint8_t* gsrc = P.src + ((int64_t)b * C + c0) * P.stride + s0;   // row 0 of this CTA, column s0
    // ------------------------------------------------------------------ F1: load the CTA's rows
    if (nload == 0) {
      if (tid == 0) mbar_arrive(bar);
    } else if (tid < nload) {
      uint32_t bytes = 0;
      for (int r = tid; r < nrows; r += nthreads) {
        const uint8_t* g = gsrc + (int64_t)r * P.stride;
        const uint32_t off = (uint32_t)(reinterpret_cast<uintptr_t>(g) & 15);
        bytes += (off + (uint32_t)tw + 15u) & ~15u;
      }
      mbar_arrive_expect_tx(bar, bytes);
      for (int r = tid; r < nrows; r += nthreads) {
        const uint8_t* g = gsrc + (int64_t)r * P.stride;
        const uint32_t off = (uint32_t)(reinterpret_cast<uintptr_t>(g) & 15);
        bulk_load(tile + (size_t)r * PW, g - off, (off + (uint32_t)tw + 15u) & ~15u, bar);
      }
    }
    mbar_wait(bar, phase);
    phase ^= 1;

    // rows rg + 4 i of one row group share the word offset of column s0 inside their shared-memory rows
    auto group_rows = [&](int rg) { return nrows > rg ? (nrows - rg + kFdRG - 1) / kFdRG : 0; };
    auto group_col0 = [&](int rg) {
      const int offw = (int)((reinterpret_cast<uintptr_t>(gsrc + (int64_t)rg * P.stride) & 15) >> 2);
      return tile + (size_t)rg * PW + offw + j;
    };

    // ------------------------------------------------------------------ F2: column statistics
    {
      uint32_t S4[4] = {0, 0, 0, 0}, Q4[4] = {0, 0, 0, 0};
      for (int rg = rg0; rg < kFdRG; rg += RG) {
      const int ni = group_rows(rg);
      const uint32_t* col = group_col0(rg);
      int i = 0;
#pragma unroll 2
      for (; i + 4 <= ni; i += 4, col += 16 * PW) {
        const uint32_t a = col[0], bb = col[4 * PW], c = col[8 * PW], d = col[12 * PW];
        const uint32_t ab_lo = prmt_b32(a, bb, 0x5140u), ab_hi = prmt_b32(a, bb, 0x7362u);
        const uint32_t cd_lo = prmt_b32(c, d, 0x5140u), cd_hi = prmt_b32(c, d, 0x7362u);
        const uint32_t t0 = prmt_b32(ab_lo, cd_lo, 0x5410u), t1 = prmt_b32(ab_lo, cd_lo, 0x7632u);
        const uint32_t t2 = prmt_b32(ab_hi, cd_hi, 0x5410u), t3 = prmt_b32(ab_hi, cd_hi, 0x7632u);
        S4[0] = __dp4a(t0, 0x01010101u, S4[0]); Q4[0] = __dp4a(t0, t0, Q4[0]);
        S4[1] = __dp4a(t1, 0x01010101u, S4[1]); Q4[1] = __dp4a(t1, t1, Q4[1]);
        S4[2] = __dp4a(t2, 0x01010101u, S4[2]); Q4[2] = __dp4a(t2, t2, Q4[2]);
        S4[3] = __dp4a(t3, 0x01010101u, S4[3]); Q4[3] = __dp4a(t3, t3, Q4[3]);
      }
      for (; i < ni; ++i, col += 4 * PW) {
        const uint32_t w = col[0];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          const uint32_t x = (w >> (8 * u)) & 0xffu;
          S4[u] += x; Q4[u] += x * x;
        }
      }
      }
      if (RG == 4) {
#pragma unroll
        for (int u = 0; u < 4; ++u) {                  // reduce over the four row groups of the warp
          S4[u] += __shfl_xor_sync(FULL, S4[u], 8);  Q4[u] += __shfl_xor_sync(FULL, Q4[u], 8);
          S4[u] += __shfl_xor_sync(FULL, S4[u], 16); Q4[u] += __shfl_xor_sync(FULL, Q4[u], 16);
        }
      }
      if (rg0 == 0) {
        reinterpret_cast<uint4*>(xS)[j] = make_uint4(S4[0], S4[1], S4[2], S4[3]);
        reinterpret_cast<uint4*>(xQ)[j] = make_uint4(Q4[0], Q4[1], Q4[2], Q4[3]);
      }
    }
    if (ncta > 1) cluster_sync_all(); else __syncthreads();

    // ------------------------------------------------------------------ F3..F5: thresholds, on chip
    // column ownership: CTA q owns word columns [q*wpc, (q+1)*wpc); thread tid < 4*wpc owns one column
    const int ocol = (int)rank * wpc * 4 + tid;
    const bool owner = tid < 4 * wpc && ocol < TsP;
    uint32_t colS = 0, colQ = 0;
    if (owner) {
      if (ncta > 1) {
        cluster_gather2(&xS[ocol], &xQ[ocol], ncta, colS, colQ);
      } else {
        colS = xS[ocol];
        colQ = xQ[ocol];
      }
    }
    const uint32_t orank = ncta > 1 ? (uint32_t)(j / wpc) : 0u;   // CTA that publishes this thread's bounds

    for (int it = 0; it < P.n_thr; ++it) {
      if (owner) {
        int lo = 0, hi = 255;
        uint32_t r = 0;
        if (ocol < tw) {
          const uint64_t V = (uint64_t)C * colQ - (uint64_t)colS * colS;
          const U8Cut cut = make_cut_u8((uint32_t)C, colS, V, P.p[it]);
          thread_bounds_u8_sqrt(cut, lo, hi);
          r = rounded_mean_u8((uint32_t)C, colS);
        }
        lo_b[ocol] = (uint8_t)lo;
        hi_b[ocol] = (uint8_t)hi;
        rr_b[ocol] = (uint8_t)r;
        uint16_t* c16 = reinterpret_cast<uint16_t*>(chk + (ocol >> 2));
        const int u = ocol & 3, slot = (u & 1) * 2 + (u >> 1);       // E.lo, O.lo, E.hi, O.hi
        c16[slot] = (uint16_t)((0x10000u - ((uint32_t)lo << 8)) & 0xffffu);
        c16[4 + slot] = (uint16_t)(lo > hi ? 0u : ((((uint32_t)(hi - lo)) << 8) | 0xffu));
      }
      if (ncta > 1) cluster_sync_all(); else __syncthreads();

      // this thread's word column: packed constants and byte bounds, pulled from the publishing CTA
      uint4 ck;
      uint32_t lo4, hi4, r4;
      if (ncta > 1) {
        ck = dsmem_ld_u128(dsmem_addr(&chk[j], orank));
        lo4 = dsmem_ld_u32(dsmem_addr(lo_b + 4 * j, orank));
        hi4 = dsmem_ld_u32(dsmem_addr(hi_b + 4 * j, orank));
        r4 = dsmem_ld_u32(dsmem_addr(rr_b + 4 * j, orank));
      } else {
        ck = chk[j];
        lo4 = reinterpret_cast<const uint32_t*>(lo_b)[j];
        hi4 = reinterpret_cast<const uint32_t*>(hi_b)[j];
        r4 = reinterpret_cast<const uint32_t*>(rr_b)[j];
      }
      const uint32_t negE = ck.x, negO = ck.y, thrE = ck.z, thrO = ck.w;
      const uint32_t chiE = 0x7fff7fffu - prmt_b32(hi4, 0u, 0x4240u), cloE = 0x80008000u - prmt_b32(lo4, 0u, 0x4240u);
      const uint32_t chiO = 0x7fff7fffu - prmt_b32(hi4, 0u, 0x4341u), cloO = 0x80008000u - prmt_b32(lo4, 0u, 0x4341u);
      // a column with an empty kept interval (lo > hi) cuts every value: no packed test can say that,
      // so such a thread takes the exact path for all its words
      const bool slow = __vcmpgtu4(lo4, hi4) != 0u;
      const bool need_stats = it + 1 < P.n_thr;

      uint32_t cnt4 = 0, sxE = 0, sxO = 0, sq[4] = {0, 0, 0, 0};   // per-column deltas of this thread, packed
      auto fix_word = [&](uint32_t* ptr, uint32_t w, int rg, int i) {
        const uint32_t m = bytes_outside_cols(w, chiE, cloE, chiO, cloO);
        if (m == 0) return;
        *ptr = (w & ~m) | (r4 & m);
        const uint32_t f = w & m;
        cnt4 += m & 0x01010101u;
        sxE += prmt_b32(f, 0u, 0x4240u);
        sxO += prmt_b32(f, 0u, 0x4341u);
        sq[0] = __dp4a(f & 0x000000ffu, f, sq[0]);
        sq[1] = __dp4a(f & 0x0000ff00u, f, sq[1]);
        sq[2] = __dp4a(f & 0x00ff0000u, f, sq[2]);
        sq[3] = __dp4a(f & 0xff000000u, f, sq[3]);
        if (P.flags) {
          uint8_t* fl = P.flags + ((int64_t)b * C + c0 + rg + kFdRG * i) * P.S + s0 + 4 * j;
#pragma unroll
          for (int u = 0; u < 4; ++u)
            if ((m >> (8 * u)) & 1u) fl[u] = 1;
        }
      };
      // Sweep first, repair afterwards: the packed test only records which four-row steps hold an outlier
      // (one bit per step); the exact repair then runs over the set bits.  A warp step covers 512 bytes,
      // so at k = 3 nearly every step has SOME lane with an outlier: repairing inside the sweep would make
      // every lane pay the repair code at every step, while the deferred loop runs max-over-lanes(popcount)
      // times (two or three for noise).
      for (int rg = rg0; rg < kFdRG; rg += RG) {
        const int ni = group_rows(rg);
        uint32_t* const colb = group_col0(rg);
        uint32_t* col = colb;
        unsigned long long hm = 0ull;
        int i = 0;
#pragma unroll 4
        for (; i + 4 <= ni; i += 4, col += 16 * PW) {
          const uint32_t w0 = col[0], w1 = col[4 * PW], w2 = col[8 * PW], w3 = col[12 * PW];
          uint32_t aO = __viaddmax_u16x2(w0, negO, 0u), aE = __viaddmax_u16x2(w0 << 8, negE, 0u);
          uint32_t bO = __viaddmax_u16x2(w1, negO, 0u), bE = __viaddmax_u16x2(w1 << 8, negE, 0u);
          aO = __viaddmax_u16x2(w2, negO, aO); aE = __viaddmax_u16x2(w2 << 8, negE, aE);
          bO = __viaddmax_u16x2(w3, negO, bO); bE = __viaddmax_u16x2(w3 << 8, negE, bE);
          aO = __vimax3_u16x2(aO, bO, thrO); aE = __vimax3_u16x2(aE, bE, thrE);
          if (aO != thrO || aE != thrE) hm |= 1ull << (i >> 2);
        }
        if (slow) hm = ~0ull;
        for (; i < ni; ++i, col += 4 * PW) fix_word(col, col[0], rg, i);
        const int nsteps = ni >> 2;
        if (nsteps < 64) hm &= (1ull << nsteps) - 1ull;
        while (hm) {
          const int st = __ffsll((long long)hm) - 1;
          hm &= hm - 1ull;
          uint32_t* c4 = colb + (size_t)st * 16 * PW;
          const uint32_t w0 = c4[0], w1 = c4[4 * PW], w2 = c4[8 * PW], w3 = c4[12 * PW];
          // usually one of the four rows holds the outlier (a narrow-band RFI channel): packed test per word
          auto hit = [&](uint32_t w) {
            return slow || __viaddmax_u16x2(w, negO, thrO) != thrO || __viaddmax_u16x2(w << 8, negE, thrE) != thrE;
          };
          if (hit(w0)) fix_word(c4, w0, rg, 4 * st);
          if (hit(w1)) fix_word(c4 + 4 * PW, w1, rg, 4 * st + 1);
          if (hit(w2)) fix_word(c4 + 8 * PW, w2, rg, 4 * st + 2);
          if (hit(w3)) fix_word(c4 + 12 * PW, w3, rg, 4 * st + 3);
        }
      }

      if (need_stats || P.counts) {
        uint32_t dS[4], dQ[4], cnt = 0;
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          const uint32_t c = (cnt4 >> (8 * u)) & 0xffu, r = (r4 >> (8 * u)) & 0xffu;
          const uint32_t sx = ((u & 1) ? sxO : sxE) >> (16 * (u >> 1)) & 0xffffu;
          dS[u] = c * r - sx;                        // modulo 2^32: the column totals stay below 2^32
          dQ[u] = c * r * r - sq[u];
          cnt += c;
        }
        if (RG == 4) {
#pragma unroll
          for (int u = 0; u < 4; ++u) {
            dS[u] += __shfl_xor_sync(FULL, dS[u], 8);  dQ[u] += __shfl_xor_sync(FULL, dQ[u], 8);
            dS[u] += __shfl_xor_sync(FULL, dS[u], 16); dQ[u] += __shfl_xor_sync(FULL, dQ[u], 16);
          }
        }
        if (need_stats && rg0 == 0) {
          reinterpret_cast<uint4*>(xS)[j] = make_uint4(dS[0], dS[1], dS[2], dS[3]);
          reinterpret_cast<uint4*>(xQ)[j] = make_uint4(dQ[0], dQ[1], dQ[2], dQ[3]);
        }
        if (P.counts) {
          cnt = __reduce_add_sync(FULL, cnt);
          if (lane == 0 && cnt) atomicAdd(&P.counts[it], (unsigned long long)cnt);
        }
      }
      if (need_stats) {
        if (ncta > 1) cluster_sync_all(); else __syncthreads();
        if (owner) {
          if (ncta > 1) {
            cluster_gather2(&xS[ocol], &xQ[ocol], ncta, colS, colQ);
          } else {
            colS += xS[ocol];
            colQ += xQ[ocol];
          }
        }
      }
    }

    // ------------------------------------------------------------------ F6: store the CTA's rows
    fence_proxy_async_smem();                       // generic-proxy writes of the fix path -> async proxy
    __syncthreads();
    {
      uint8_t* gdst = P.dst + ((int64_t)b * C + c0) * P.stride + s0;
      bool issued = false;
      for (int r = tid; r < nrows; r += nthreads) {
        const uint32_t off = (uint32_t)(reinterpret_cast<uintptr_t>(gsrc + (int64_t)r * P.stride) & 15);
        const uint8_t* srow = reinterpret_cast<const uint8_t*>(tile + (size_t)r * PW) + off;   // column s0
        uint8_t* gd = gdst + (int64_t)r * P.stride;
        // src and dst share their 16-byte phase (checked by the host), so the aligned interior of the
        // destination is aligned in shared memory too
        int h = (int)((16u - off) & 15u);
        if (h > tw) h = tw;
        const int body = (tw - h) & ~15;
        if (body > 0) {
          bulk_store(gd + h, srow + h, (uint32_t)body);
          issued = true;
        }
        int i = 0;
        for (; i + 4 <= h; i += 4) *reinterpret_cast<uint32_t*>(gd + i) = *reinterpret_cast<const uint32_t*>(srow + i);
        for (; i < h; ++i) gd[i] = srow[i];
        i = h + body;
        for (; i + 4 <= tw; i += 4) *reinterpret_cast<uint32_t*>(gd + i) = *reinterpret_cast<const uint32_t*>(srow + i);
        for (; i < tw; ++i) gd[i] = srow[i];
      }
      if (issued) {
        bulk_commit();
        bulk_wait_read<0>();                        // the rows may be overwritten after this
      }
    }
    __syncthreads();
  }
  bulk_wait_all<0>();
  if (ncta > 1) cluster_sync_all();                 // no CTA leaves while a peer may still read its shared memory
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
