// fd_u8_stream.cuh -- frequency-domain sigma cut (FDSC, Fig. 3) for uint8 dynamic spectra:
// the streaming kernel (8f NEXT-1: the per-bin mean correction of PAPER.md:102,126).
// Reachable as variant 16 only: its one-bin form has been overtaken by fd_u8_quad.cuh, which keeps this file's
// geometry, ring and ticket scheme and changes the division of labour, its binned form by fd_u8_qbin.cuh, which
// streams the tile once per threshold step instead of repairing candidate blocks.  Both successors
// use this file's parameter block, box geometry and helpers.
//
// A tile is ALL channels x 128 consecutive samples of one beam.  Unlike a kernel that keeps the tile resident in
// shared memory, this one streams it ONCE through small per-warp rings and keeps, per thread, only
//   * the exact column sums (S, Q) of its 4 sample columns, and
//   * one SUMMARY per 4-channel x 4-sample block it has seen: the largest and the smallest of its 16 bytes
//     (two bytes per 16 data bytes, held in registers).
// A cut with kept interval [lo_c, hi_c] per column can only touch a block whose max exceeds the smallest hi or
// whose min is below the largest lo of its 4 columns, so a threshold iteration is a packed test of the summaries
// (a few instructions per thread) followed by an exact repair of the few candidate blocks, which are re-read
// from and written back to global memory (they are still in L1/L2).  In place nothing else is written: a sample
// that is not replaced keeps its bytes (HBM sees one read per sample and one sector write per replaced sample);
// out of place every word is copied to the destination in the statistics pass (one read + one write per sample).
//
//   F1  warp w owns RW = C / 16 rows of one 16-byte alignment class (row mod 4 = w mod 4: rows 4 apart are
//       4 * pitch bytes apart, a multiple of 16, so a class is a 2-D tensor a TMA tensor map can describe even on
//       the dense 12500-byte pitch).  It streams them as boxes of 8 rows x 144 bytes (the 16-byte aligned superset
//       of the 128 columns) through a ring of kSlots boxes, one mbarrier each: kSlots - 1 boxes are always in
//       flight per warp, also across tile boundaries, and the ring is free again as soon as the statistics
//       pass is over, so the next tile's first boxes land while this tile is being thresholded.
//   F2  lane = word column (4 samples).  Per block of 4 rows: PRMT 4x4 byte transposes + IDP.4A give exact column
//       sums / sums of squares; VIMNMX3.U16x2 gives the block summary.  Warps meet in shared-memory accumulators.
//   F3  one thread per column: exact kept interval in closed form (integer square root), replacement value.
//       With bins (PAPER.md:102 step 1): per-bin sums S_b, V = nb Q - sum_b S_b^2, T = isqrt(floor(p^2 nb V /
//       (2^32 C))), and per (bin, column) lo = ceil((S_b - T) / nb), hi = floor((S_b + T) / nb), r = rounded S_b / nb.
//   F4  packed summary test -> candidate blocks -> exact per-byte masks, replace, column (and bin) deltas.
//   F5  next threshold from the updated sums; summaries of repaired blocks are left as they were (conservative:
//       such a block is simply examined again).   F6  see above: nothing left to do.
#pragma once

#include <cuda.h>   // CUtensorMap (types only: the encoder is fetched through the runtime, no -lcuda)

#include "common.cuh"
#include "packed.cuh"

namespace rfim {

constexpr int kFsCols = 128;                       // samples per tile
constexpr int kFsPitchW = 36;                      // words per row in a ring box: 144 bytes
constexpr int kFsBoxRows = 8;                      // class rows per box (two blocks of 4)
constexpr int kFsBoxWords = kFsBoxRows * kFsPitchW;   // 288 words = 1152 bytes = 9 * 128
constexpr int kFsWarps = 16;
constexpr int kFsThreads = 32 * kFsWarps;
constexpr int kFsMaxBins = 256;

struct FdStreamMaps {
  CUtensorMap src[4];                              // one per alignment class (row mod 4)
};

struct FdStreamParams {
  const uint8_t* src;
  uint8_t* dst;
  int64_t stride;
  int beams, C, S;                                 // beams of THIS launch (the tensor maps cover the whole buffer)
  int beam0;                                       // first beam of this launch inside the buffer
  int n_thr;
  uint32_t p[16];
  uint8_t* flags;                                  // optional, dense [buffer beams][C][S]
  unsigned long long* counts;
  int tiles_per_beam;
  int64_t total_tiles;
  int off[4];                                      // byte offset of column s0 inside a box of class k
  uint32_t invC;                                   // ceil(2^32 / C)
  int nb, nbins;                                   // binned: channels per bin (multiple of 16), bins
  uint32_t inv_nb, inv_2nb;                        // ceil(2^32 / nb), ceil(2^32 / (2 nb))
  int off_dst[4];                                  // fd_u8_qbin: the same offsets for the destination's tensor maps
  unsigned int* ticket;                            // tile dispenser of this launch (device, zero before the launch)
};

// shared memory of one CTA: [rings: 16 warps x kSlots boxes][FsCtrl][binned: binS[2][nbins][64], lo/hi/r[nbins][128]]
struct __align__(16) FsCtrl {
  uint32_t acc[2][2 * kFsCols];                    // [buffer][S of 128 columns | Q of 128 columns]
  uint8_t lo[kFsCols], hi[kFsCols], rr[kFsCols];
  uint32_t T[kFsCols];                             // binned: per-column threshold on |nb x - S_b|
  uint64_t full[kFsWarps][4];                      // ring mbarriers
  int tk[3][3];                                    // tile tickets handed to this CTA: {tile, beam, tile in beam}
};
__host__ __device__ inline size_t fd_stream_smem_bytes(int slots, int nbins_or_0) {
  size_t b = (size_t)kFsWarps * slots * kFsBoxWords * 4 + sizeof(FsCtrl);
  if (nbins_or_0 > 0) b += (size_t)2 * nbins_or_0 * (kFsCols / 2) * 4 + (size_t)3 * nbins_or_0 * kFsCols;
  return b;
}

__device__ __forceinline__ void fs_tma_load_2d(void* smem_dst, const CUtensorMap* map, int x, int y, uint64_t* bar) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
      ::"r"(smem_addr(smem_dst)), "l"(reinterpret_cast<uint64_t>(map)), "r"(x), "r"(y), "r"(smem_addr(bar))
      : "memory");
}
__device__ __forceinline__ void fs_prefetch_desc(const CUtensorMap* map) {
  asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(map)) : "memory");
}
__device__ __forceinline__ void fs_red_add(uint32_t* p, uint32_t v) {
  asm volatile("red.shared.add.u32 [%0], %1;" ::"r"(smem_addr(p)), "r"(v) : "memory");
}
// largest / smallest of the four bytes of a word
__device__ __forceinline__ uint32_t fs_max4(uint32_t w) {
  const uint32_t a = max(w & 0xffu, (w >> 8) & 0xffu), b = max((w >> 16) & 0xffu, w >> 24);
  return max(a, b);
}
__device__ __forceinline__ uint32_t fs_min4(uint32_t w) {
  const uint32_t a = min(w & 0xffu, (w >> 8) & 0xffu), b = min((w >> 16) & 0xffu, w >> 24);
  return min(a, b);
}
// floor(a / n) for a < 2^62 from a double estimate, corrected with exact integer checks
__device__ __forceinline__ uint64_t fs_div_u64(uint64_t a, uint32_t n) {
  uint64_t q = (uint64_t)((double)a / (double)n);
  while (q * n > a) --q;
  while (a - q * n >= n) ++q;
  return q;
}

// NCH = boxes per warp and tile (C = 128 * NCH channels); kBinned: per-bin mean correction; kCopy: out of place
template <int NCH, int kSlots, bool kBinned, bool kCopy>
__global__ void __launch_bounds__(kFsThreads, 2) fd_u8_stream_kernel(const __grid_constant__ FdStreamMaps maps,
                                                                     const FdStreamParams P) {
  extern __shared__ __align__(128) uint8_t smem[];
  constexpr int RW = NCH * kFsBoxRows;               // class rows per warp
  constexpr int NREG = (2 * NCH + 3) / 4;            // summary registers: 2 blocks per box, 4 bytes per register
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int cls = warp & 3, g = warp >> 2;
  const int C = P.C;
  uint32_t* const ring = reinterpret_cast<uint32_t*>(smem) + (size_t)warp * kSlots * kFsBoxWords;
  FsCtrl* const K = reinterpret_cast<FsCtrl*>(smem + (size_t)kFsWarps * kSlots * kFsBoxWords * 4);
  uint32_t* const binS = reinterpret_cast<uint32_t*>(K + 1);                        // [2][nbins][64]: two columns per word
  uint8_t* const loB = reinterpret_cast<uint8_t*>(binS + 2 * P.nbins * (kFsCols / 2));   // [nbins][128]
  uint8_t* const hiB = loB + P.nbins * kFsCols;
  uint8_t* const rB = hiB + P.nbins * kFsCols;
  uint64_t* const full = &K->full[warp][0];

  if (tid == 0) {
#pragma unroll
    for (int k = 0; k < 4; ++k) fs_prefetch_desc(&maps.src[k]);
  }
  if (lane == 0) {
#pragma unroll
    for (int s = 0; s < kSlots; ++s) mbar_init(&full[s], 1);
    fence_mbar_init();
  }
  for (int i = tid; i < 4 * kFsCols; i += kFsThreads) (&K->acc[0][0])[i] = 0;
  if (kBinned)
    for (int i = tid; i < 2 * P.nbins * (kFsCols / 2); i += kFsThreads) binS[i] = 0;
  __syncthreads();

  // box `c` of a tile of this warp: rows [g RW + 8 c, + 8) of class cls of the tile's beam (y0 = the warp's first
  // class row of that beam), x = the tile's first column
  auto issue = [&](int s0, int y0, int c, int slot) {   // one lane
    mbar_arrive_expect_tx(&full[slot], kFsBoxWords * 4u);
    fs_tma_load_2d(ring + slot * kFsBoxWords, &maps.src[cls], s0, y0 + kFsBoxRows * c, &full[slot]);
  };
  // Tiles are handed out by a ticket counter, in order, two tickets ahead (the ring prefetches into the next tile).
  // With a fixed stride the CTAs drift apart and the 64-byte DRAM atoms that neighbouring tiles share (a box row is
  // the 144-byte superset of 128 columns of a 4-byte aligned row) are fetched twice: 18.7 GB of DRAM reads for a
  // 9.2 GB batch.  Tickets keep neighbouring tiles in flight at the same time, so the second request hits L2.
  auto take_ticket = [&](int slot_) {                 // one thread
    const unsigned int t = atomicAdd(P.ticket, 1u);
    const unsigned int tb = t / (unsigned int)P.tiles_per_beam;
    K->tk[slot_][0] = (int)min(t, 0x7fffffffu);
    K->tk[slot_][1] = (int)tb;
    K->tk[slot_][2] = (int)(t - tb * (unsigned int)P.tiles_per_beam);
  };
  if (tid == 0) { take_ticket(0); take_ticket(1); }
  __syncthreads();
  int64_t cur_t = K->tk[0][0];
  int cur_b = K->tk[0][1], cur_q = K->tk[0][2];
  int64_t nxt_t = K->tk[1][0];
  int nxt_b = K->tk[1][1], nxt_q = K->tk[1][2];
  const int ywarp = g * RW;                           // + (beam * C) / 4: the warp's first class row of a beam
  const int cq = C >> 2;
  if (lane == 0 && cur_t < P.total_tiles) {
#pragma unroll
    for (int c = 0; c < kSlots; ++c) {
      // NCH >= kSlots is guaranteed by the host
      issue(cur_q * kFsCols, (P.beam0 + cur_b) * cq + ywarp, c, c);
    }
  }
  // binned: bit s of binend <=> this thread's block s is the last block of its bin; bin0 = bin of block 0.
  // (a block is 4 class rows = 16 channels; nb is a multiple of 16 and bins do not straddle warps: host-checked)
  uint32_t binend = 0;
  int bin0 = 0;
  if (kBinned) {
    const int bpb = P.nb >> 4;                        // blocks per bin
    bin0 = (4 * g * RW) / P.nb;
    for (int s = 0; s < 2 * NCH; ++s)
      if ((s + 1) % bpb == 0) binend |= 1u << s;
  }

  uint32_t phases = 0;                                // one parity bit per ring slot
  int slot = 0;
  int buf = 0;                                        // accumulator buffer of the next exchange
  int bsel = 0;                                       // binned: bin-sum buffer of this tile
  uint32_t colS = 0, colQ = 0;                        // column owners (tid < 128): exact totals, kept across iterations
  const int offw = P.off[cls] >> 2;                   // word offset of column s0 inside a box row

  while (cur_t < P.total_tiles) {
    const int b = P.beam0 + cur_b;
    const int s0 = cur_q * kFsCols;
    const bool have_next = nxt_t < P.total_tiles;
    const int nxt_s0 = nxt_q * kFsCols, nxt_y0 = (P.beam0 + nxt_b) * cq + ywarp, cur_y0 = b * cq + ywarp;
    const int tw = min(kFsCols, P.S - s0);            // valid columns of this tile
    const int nvalid = tw - 4 * lane;                 // valid bytes of this lane's word (>= 4: all)
    // row 0 of this warp's rows is channel 4 * (g RW) + cls; consecutive class rows are 4 channels apart
    uint8_t* const dwarp = P.dst + ((int64_t)b * C + 4 * (g * RW) + cls) * P.stride + s0 + 4 * lane;
    const int64_t rstep = 4 * P.stride;
    uint32_t* const bS = binS + bsel * P.nbins * (kFsCols / 2);

    // ------------------------------------------------------------------ F1 + F2: stream the rows once
    uint32_t MX[NREG], MN[NREG];
#pragma unroll
    for (int i = 0; i < NREG; ++i) { MX[i] = 0u; MN[i] = 0u; }
    uint32_t S4[4] = {0, 0, 0, 0}, Q4[4] = {0, 0, 0, 0};
    uint32_t B4[4] = {0, 0, 0, 0};                    // binned: sums of the current bin
    int fbin = bin0;                                  // binned: the bin being summed
#pragma unroll
    for (int c = 0; c < NCH; ++c) {
      mbar_wait(&full[slot], (phases >> slot) & 1u);
      phases ^= 1u << slot;
      const uint32_t* rowp = ring + slot * kFsBoxWords + offw + lane;
      uint32_t w[kFsBoxRows];
#pragma unroll
      for (int j = 0; j < kFsBoxRows; ++j) w[j] = rowp[j * kFsPitchW];
      if (kCopy) {
        uint8_t* gd = dwarp + (int64_t)(kFsBoxRows * c) * rstep;
        if (nvalid >= 4) {
#pragma unroll
          for (int j = 0; j < kFsBoxRows; ++j) *reinterpret_cast<uint32_t*>(gd + j * rstep) = w[j];
        } else if (nvalid > 0) {
          for (int j = 0; j < kFsBoxRows; ++j)
            for (int u = 0; u < nvalid; ++u) gd[j * rstep + u] = (uint8_t)(w[j] >> (8 * u));
        }
      }
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        const uint32_t a = w[4 * h], bb = w[4 * h + 1], cc = w[4 * h + 2], d = w[4 * h + 3];
        const uint32_t ab_lo = prmt_b32(a, bb, 0x5140u), ab_hi = prmt_b32(a, bb, 0x7362u);
        const uint32_t cd_lo = prmt_b32(cc, d, 0x5140u), cd_hi = prmt_b32(cc, d, 0x7362u);
        const uint32_t t0 = prmt_b32(ab_lo, cd_lo, 0x5410u), t1 = prmt_b32(ab_lo, cd_lo, 0x7632u);
        const uint32_t t2 = prmt_b32(ab_hi, cd_hi, 0x5410u), t3 = prmt_b32(ab_hi, cd_hi, 0x7632u);
        if (kBinned) {
          B4[0] = __dp4a(t0, 0x01010101u, B4[0]); B4[1] = __dp4a(t1, 0x01010101u, B4[1]);
          B4[2] = __dp4a(t2, 0x01010101u, B4[2]); B4[3] = __dp4a(t3, 0x01010101u, B4[3]);
        } else {
          S4[0] = __dp4a(t0, 0x01010101u, S4[0]); S4[1] = __dp4a(t1, 0x01010101u, S4[1]);
          S4[2] = __dp4a(t2, 0x01010101u, S4[2]); S4[3] = __dp4a(t3, 0x01010101u, S4[3]);
        }
        Q4[0] = __dp4a(t0, t0, Q4[0]); Q4[1] = __dp4a(t1, t1, Q4[1]);
        Q4[2] = __dp4a(t2, t2, Q4[2]); Q4[3] = __dp4a(t3, t3, Q4[3]);
        const uint32_t e = group_summary(make_uint4(a, bb, cc, d));     // byte 1 = max, byte 0 = min
        constexpr uint32_t selx[4] = {0x3215u, 0x3250u, 0x3510u, 0x5210u};
        constexpr uint32_t seln[4] = {0x3214u, 0x3240u, 0x3410u, 0x4210u};
        const int s = 2 * c + h;                      // block index of this thread
        MX[s >> 2] = prmt(MX[s >> 2], e, selx[s & 3]);
        MN[s >> 2] = prmt(MN[s >> 2], e, seln[s & 3]);
        if (kBinned && ((binend >> s) & 1u)) {       // warp-uniform: the bin ends with this block
          fs_red_add(&bS[fbin * (kFsCols / 2) + 2 * lane], B4[0] | (B4[1] << 16));
          fs_red_add(&bS[fbin * (kFsCols / 2) + 2 * lane + 1], B4[2] | (B4[3] << 16));
          B4[0] = 0; B4[1] = 0; B4[2] = 0; B4[3] = 0;
          ++fbin;
        }
      }
      // Refill the box only now: the statistics above have CONSUMED the eight words, so every lane's shared-memory
      // loads have completed.  (Re-arming right after the loads were merely issued lets the asynchronous copy
      // overtake them once the refill hits L2: a write-after-read hazard that showed up as rare wrong column sums.)
      __syncwarp();
      if (lane == 0) {
        if (c + kSlots < NCH) issue(s0, cur_y0, c + kSlots, slot);                    // compile-time branch
        else if (have_next) issue(nxt_s0, nxt_y0, c + kSlots - NCH, slot);
      }
      slot = (slot + 1 == kSlots) ? 0 : slot + 1;
    }
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      if (!kBinned) fs_red_add(&K->acc[buf][4 * lane + u], S4[u]);
      fs_red_add(&K->acc[buf][kFsCols + 4 * lane + u], Q4[u]);
    }

    // ------------------------------------------------------------------ F3..F5: thresholds
    int64_t nn_t = 0x7fffffff;
    int nn_b = 0, nn_q = 0;
    for (int it = 0; it < P.n_thr; ++it) {
      const bool first = it == 0;
      const bool need_stats = it + 1 < P.n_thr;
      // ---- exchange: accumulators -> column owners -> bounds for everybody
      __syncthreads();                                                // A: accumulators (and bin sums) complete
      if (first && tid == kFsThreads - 1) take_ticket(2);             // the tile after the next one
      if (tid < kFsCols) {
        const uint32_t q = K->acc[buf][kFsCols + tid];
        if (first) colQ = q; else colQ += q;                          // deltas are modulo 2^32
        if (!kBinned) {
          const uint32_t s = K->acc[buf][tid];
          if (first) colS = s; else colS += s;
          int lo = 0, hi = 255;
          uint32_t r = 0;
          if (tid < tw) {
            const uint64_t V = (uint64_t)C * colQ - (uint64_t)colS * colS;
            const U8Cut cut = make_cut_u8((uint32_t)C, colS, V, P.p[it]);
            thread_bounds_u8_sqrt32(cut, P.invC, lo, hi, r);
          }
          K->lo[tid] = (uint8_t)lo;
          K->hi[tid] = (uint8_t)hi;
          K->rr[tid] = (uint8_t)r;
        } else {
          // V = nb Q - sum_b S_b^2;  T = isqrt(floor(p^2 nb V / (2^32 C)))
          uint64_t ss = 0;
          const int sh = (tid & 1) * 16;
          for (int bn = 0; bn < P.nbins; ++bn) {
            const uint32_t sb = (bS[bn * (kFsCols / 2) + (tid >> 1)] >> sh) & 0xffffu;
            ss += (uint64_t)sb * sb;
          }
          const uint64_t V = (uint64_t)P.nb * colQ - ss;
          const uint64_t nbV = (uint64_t)P.nb * V;                    // < 2^45 (nb <= 256, C <= 4096)
          const uint64_t p2 = (uint64_t)P.p[it] * P.p[it];
          const uint64_t xh = __umul64hi(p2, nbV), xl = p2 * nbV;     // p^2 nb V < 2^93
          const uint64_t Y = (xh << 32) | (xl >> 32);                 // floor(p^2 nb V / 2^32) < 2^61
          const uint64_t W = fs_div_u64(Y, (uint32_t)C);
          uint64_t T = (uint64_t)__dsqrt_rd((double)W);
          while (T * T > W) --T;
          while ((T + 1) * (T + 1) <= W) ++T;
          K->T[tid] = tid < tw ? (uint32_t)min(T, (uint64_t)0xffffu) : 0xffffu;   // |nb x - S_b| <= 255 nb < 65535
        }
      }
      if (kBinned) {
        __syncthreads();                                              // A2: thresholds published
        for (int idx = tid; idx < P.nbins * kFsCols; idx += kFsThreads) {
          const int bn = idx >> 7, col = idx & (kFsCols - 1);
          const uint32_t sb = (bS[bn * (kFsCols / 2) + (col >> 1)] >> ((col & 1) * 16)) & 0xffffu;
          const uint32_t T = K->T[col];
          uint32_t hi = div_floor_u32(sb + T, (uint32_t)P.nb, P.inv_nb);
          if (hi > 255u) hi = 255u;
          uint32_t lo = sb > T ? div_floor_u32(sb - T + (uint32_t)P.nb - 1u, (uint32_t)P.nb, P.inv_nb) : 0u;
          if (lo > hi) { lo = 1; hi = 0; }
          loB[idx] = (uint8_t)lo;
          hiB[idx] = (uint8_t)hi;
          rB[idx] = (uint8_t)div_floor_u32(2u * sb + (uint32_t)P.nb, 2u * (uint32_t)P.nb, P.inv_2nb);
        }
      }
      __syncthreads();                                                // B: bounds published
      if (first) { nn_t = K->tk[2][0]; nn_b = K->tk[2][1]; nn_q = K->tk[2][2]; }
      if (tid < 2 * kFsCols) K->acc[buf][tid] = 0;                    // nobody reads this buffer any more
      buf ^= 1;
      if (kBinned && first) {                                         // the other bin-sum buffer is idle until the next tile
        uint32_t* const other = binS + (bsel ^ 1) * P.nbins * (kFsCols / 2);
        for (int i = tid; i < P.nbins * (kFsCols / 2); i += kFsThreads) other[i] = 0;
      }

      // ---- candidate blocks from the summaries
      uint32_t hm = 0;
      uint32_t lo4 = 0, hi4 = 0, r4 = 0;
      if (!kBinned) {
        lo4 = reinterpret_cast<const uint32_t*>(K->lo)[lane];
        hi4 = reinterpret_cast<const uint32_t*>(K->hi)[lane];
        r4 = reinterpret_cast<const uint32_t*>(K->rr)[lane];
        const uint32_t cab2 = (0x7fffu - fs_min4(hi4)) * 0x00010001u;
        const uint32_t cbe2 = (0x7fffu + fs_max4(lo4)) * 0x00010001u;
#pragma unroll
        for (int i = 0; i < NREG; ++i) {
          const uint32_t m = bytes_above(MX[i], cab2) | bytes_below(MN[i], cbe2);
          hm |= (((m & 0x01010101u) * 0x01020408u) >> 24) << (4 * i);
        }
      } else {
        // the blocks of one bin share their bounds
        int bin = bin0;
        uint32_t himin = 0, lomax = 0;
        bool fresh = true;
#pragma unroll
        for (int s = 0; s < 2 * NCH; ++s) {
          if (fresh) {                                                // warp-uniform
            himin = fs_min4(reinterpret_cast<const uint32_t*>(hiB)[bin * (kFsCols / 4) + lane]);
            lomax = fs_max4(reinterpret_cast<const uint32_t*>(loB)[bin * (kFsCols / 4) + lane]);
          }
          const uint32_t mx = (MX[s >> 2] >> (8 * (s & 3))) & 0xffu, mn = (MN[s >> 2] >> (8 * (s & 3))) & 0xffu;
          if (mx > himin || mn < lomax) hm |= 1u << s;
          fresh = (binend >> s) & 1u;
          bin += fresh ? 1 : 0;
        }
      }
      if (2 * NCH < 32) hm &= (1u << ((2 * NCH) & 31)) - 1u;

      // ---- exact repair of the candidate blocks, through global memory (L1 / L2)
      uint32_t cnt4 = 0, sxE = 0, sxO = 0, sq[4] = {0, 0, 0, 0};      // per-column deltas of this thread, packed
      uint32_t rq[4] = {0, 0, 0, 0};                                  // binned: sum of r^2 over the replaced bytes
      uint32_t chiE = 0, cloE = 0, chiO = 0, cloO = 0;
      if (!kBinned) {
        chiE = 0x7fff7fffu - prmt_b32(hi4, 0u, 0x4240u); cloE = 0x80008000u - prmt_b32(lo4, 0u, 0x4240u);
        chiO = 0x7fff7fffu - prmt_b32(hi4, 0u, 0x4341u); cloO = 0x80008000u - prmt_b32(lo4, 0u, 0x4341u);
      }
      // Packed pre-test of a word against its four columns' kept intervals (two VIADDMNMX.U16x2): with neg = -lo and
      // thr = hi - lo in the high byte of a u16 lane (low byte 0xff), (x + neg) mod 2^16 > thr <=> x outside [lo, hi].
      // A column with an empty kept interval (lo > hi) cuts every value, which the packed form cannot say: `slow`.
      uint32_t negE = 0, negO = 0, thrE = 0, thrO = 0;
      bool slow = false;
      auto packed_bounds = [&]() {
        const uint32_t loE = prmt_b32(lo4, 0u, 0x2404u), loO = prmt_b32(lo4, 0u, 0x3414u);   // lo << 8 per u16 lane
        const uint32_t hiE = prmt_b32(hi4, 0u, 0x2404u), hiO = prmt_b32(hi4, 0u, 0x3414u);
        negE = __vsub2(0u, loE); negO = __vsub2(0u, loO);
        thrE = __vsub2(hiE, loE) | 0x00ff00ffu; thrO = __vsub2(hiO, loO) | 0x00ff00ffu;
        slow = __vcmpgtu4(lo4, hi4) != 0u;
      };
      auto word_hit = [&](uint32_t wv) {
        return slow || __viaddmax_u16x2(wv, negO, thrO) != thrO || __viaddmax_u16x2(wv << 8, negE, thrE) != thrE;
      };
      if (!kBinned) packed_bounds();
      if (nvalid <= 0) hm = 0;
      // One word of a candidate block: exact per-byte mask, replace in global memory, column (and bin) deltas.
      uint32_t bsx01 = 0, bsx23 = 0;                                  // binned: packed signed deltas of the bin sums
      auto fix_word = [&](uint32_t wv, uint8_t* gw, int ch, int nv) -> uint32_t {
        uint32_t m = bytes_outside_cols(wv, chiE, cloE, chiO, cloO);
        if (nv < 4) m &= (1u << (8 * nv)) - 1u;
        if (m == 0) return wv;
        const uint32_t nw = (wv & ~m) | (r4 & m);
        if (nv >= 4) {
          *reinterpret_cast<uint32_t*>(gw) = nw;
        } else {
          for (int u = 0; u < nv; ++u) gw[u] = (uint8_t)(nw >> (8 * u));
        }
        const uint32_t f = wv & m;
        cnt4 += m & 0x01010101u;
        sq[0] = __dp4a(f & 0x000000ffu, f, sq[0]);
        sq[1] = __dp4a(f & 0x0000ff00u, f, sq[1]);
        sq[2] = __dp4a(f & 0x00ff0000u, f, sq[2]);
        sq[3] = __dp4a(f & 0xff000000u, f, sq[3]);
        if (!kBinned) {
          sxE += prmt_b32(f, 0u, 0x4240u);
          sxO += prmt_b32(f, 0u, 0x4341u);
        } else {
          // r - x per replaced byte, two columns per word: plain 32-bit arithmetic is exact here because the
          // bin sums are back inside their 16-bit fields once all deltas of the iteration are in
          const uint32_t rm = r4 & m;
          bsx01 += (rm & 0xffu) - (f & 0xffu) + ((((rm >> 8) & 0xffu) - ((f >> 8) & 0xffu)) << 16);
          bsx23 += ((rm >> 16) & 0xffu) - ((f >> 16) & 0xffu) + (((rm >> 24) - (f >> 24)) << 16);
          rq[0] = __dp4a(rm & 0x000000ffu, rm, rq[0]);                // r differs from bin to bin
          rq[1] = __dp4a(rm & 0x0000ff00u, rm, rq[1]);
          rq[2] = __dp4a(rm & 0x00ff0000u, rm, rq[2]);
          rq[3] = __dp4a(rm & 0xff000000u, rm, rq[3]);
        }
        if (P.flags) {
          uint8_t* fl = P.flags + ((int64_t)b * C + ch) * P.S + s0 + 4 * lane;
#pragma unroll
          for (int u = 0; u < 4; ++u)
            if ((m >> (8 * u)) & 1u) fl[u] = 1;
        }
        return nw;
      };
      if (nvalid >= 4) {
        // The next candidate's four words are requested before the current block is examined: the blocks are
        // distinct, and a warp's trip count is the largest candidate count among its lanes, so the L2 round trip
        // is what a trip costs otherwise.
        uint32_t wn[4] = {0, 0, 0, 0};
        int sn = -1;
        if (hm) {
          sn = __ffs(hm) - 1;
          hm &= hm - 1;
          const uint8_t* gp = dwarp + (int64_t)(4 * sn) * rstep;
#pragma unroll
          for (int i = 0; i < 4; ++i) wn[i] = *reinterpret_cast<const uint32_t*>(gp + i * rstep);
        }
        while (sn >= 0) {
          const int s = sn;
          const uint32_t w0 = wn[0], w1 = wn[1], w2 = wn[2], w3 = wn[3];
          sn = -1;
          if (hm) {
            sn = __ffs(hm) - 1;
            hm &= hm - 1;
            const uint8_t* gp = dwarp + (int64_t)(4 * sn) * rstep;
#pragma unroll
            for (int i = 0; i < 4; ++i) wn[i] = *reinterpret_cast<const uint32_t*>(gp + i * rstep);
          }
          int bin = 0;
          if (kBinned) {
            bin = bin0 + __popc(binend & ((1u << s) - 1u));           // bins that ended before block s
            hi4 = reinterpret_cast<const uint32_t*>(hiB)[bin * (kFsCols / 4) + lane];
            lo4 = reinterpret_cast<const uint32_t*>(loB)[bin * (kFsCols / 4) + lane];
            r4 = reinterpret_cast<const uint32_t*>(rB)[bin * (kFsCols / 4) + lane];
            chiE = 0x7fff7fffu - prmt_b32(hi4, 0u, 0x4240u); cloE = 0x80008000u - prmt_b32(lo4, 0u, 0x4240u);
            chiO = 0x7fff7fffu - prmt_b32(hi4, 0u, 0x4341u); cloO = 0x80008000u - prmt_b32(lo4, 0u, 0x4341u);
            bsx01 = 0; bsx23 = 0;
            packed_bounds();
          }
          const bool h0 = word_hit(w0), h1 = word_hit(w1), h2 = word_hit(w2), h3 = word_hit(w3);
          if (h0 | h1 | h2 | h3) {
            uint8_t* gp = dwarp + (int64_t)(4 * s) * rstep;
            const int ch = 4 * (g * RW + 4 * s) + cls;
            uint32_t n0 = w0, n1 = w1, n2 = w2, n3 = w3;
            if (h0) n0 = fix_word(w0, gp, ch, 4);
            if (h1) n1 = fix_word(w1, gp + rstep, ch + 4, 4);
            if (h2) n2 = fix_word(w2, gp + 2 * rstep, ch + 8, 4);
            if (h3) n3 = fix_word(w3, gp + 3 * rstep, ch + 12, 4);
            if (kBinned && need_stats && (bsx01 | bsx23)) {
              fs_red_add(&bS[bin * (kFsCols / 2) + 2 * lane], bsx01);
              fs_red_add(&bS[bin * (kFsCols / 2) + 2 * lane + 1], bsx23);
            }
            if (need_stats) {
              // a later iteration should not examine this block again for what has just been replaced: refresh its
              // summary (byte s & 3 of register s >> 2; the register index is resolved by predication)
              const uint32_t e = group_summary(make_uint4(n0, n1, n2, n3));
              const int sh = 4 * (s & 3);
              const uint32_t selx = (0x3210u & ~(0xfu << sh)) | (0x5u << sh);
              const uint32_t seln = (0x3210u & ~(0xfu << sh)) | (0x4u << sh);
#pragma unroll
              for (int i = 0; i < NREG; ++i)
                if ((s >> 2) == i) { MX[i] = prmt(MX[i], e, selx); MN[i] = prmt(MN[i], e, seln); }
            }
          }
        }
      } else {
        // the last word of a row with 1..3 valid bytes: byte-granular loads and stores
        while (hm) {
          const int s = __ffs(hm) - 1;
          hm &= hm - 1;
          int bin = 0;
          if (kBinned) {
            bin = bin0 + __popc(binend & ((1u << s) - 1u));
            hi4 = reinterpret_cast<const uint32_t*>(hiB)[bin * (kFsCols / 4) + lane];
            lo4 = reinterpret_cast<const uint32_t*>(loB)[bin * (kFsCols / 4) + lane];
            r4 = reinterpret_cast<const uint32_t*>(rB)[bin * (kFsCols / 4) + lane];
            chiE = 0x7fff7fffu - prmt_b32(hi4, 0u, 0x4240u); cloE = 0x80008000u - prmt_b32(lo4, 0u, 0x4240u);
            chiO = 0x7fff7fffu - prmt_b32(hi4, 0u, 0x4341u); cloO = 0x80008000u - prmt_b32(lo4, 0u, 0x4341u);
            bsx01 = 0; bsx23 = 0;
          }
          uint8_t* gp = dwarp + (int64_t)(4 * s) * rstep;
          for (int i = 0; i < 4; ++i) {
            uint32_t wv = 0;
            for (int u = 0; u < nvalid; ++u) wv |= (uint32_t)gp[i * rstep + u] << (8 * u);
            fix_word(wv, gp + i * rstep, 4 * (g * RW + 4 * s + i) + cls, nvalid);
          }
          if (kBinned && need_stats && (bsx01 | bsx23)) {
            fs_red_add(&bS[bin * (kFsCols / 2) + 2 * lane], bsx01);
            fs_red_add(&bS[bin * (kFsCols / 2) + 2 * lane + 1], bsx23);
          }
        }
      }
      if ((need_stats || P.counts) && __any_sync(FULL, cnt4 != 0u)) {
        uint32_t cnt = 0;
        if (cnt4) {
#pragma unroll
          for (int u = 0; u < 4; ++u) {
            const uint32_t c = (cnt4 >> (8 * u)) & 0xffu;
            cnt += c;
            if (!kBinned && need_stats && c) {                        // modulo 2^32: the column totals stay below 2^32
              const uint32_t r = (r4 >> (8 * u)) & 0xffu;
              const uint32_t sx = ((u & 1) ? sxO : sxE) >> (16 * (u >> 1)) & 0xffffu;
              fs_red_add(&K->acc[buf][4 * lane + u], c * r - sx);
              fs_red_add(&K->acc[buf][kFsCols + 4 * lane + u], c * r * r - sq[u]);
            }
            if (kBinned && need_stats && c) fs_red_add(&K->acc[buf][kFsCols + 4 * lane + u], rq[u] - sq[u]);
          }
        }
        if (P.counts) {
          cnt = __reduce_add_sync(FULL, cnt);
          if (lane == 0 && cnt) atomicAdd(&P.counts[it], (unsigned long long)cnt);
        }
      }
    }
    bsel ^= 1;
    cur_t = nxt_t; cur_b = nxt_b; cur_q = nxt_q;
    nxt_t = nn_t; nxt_b = nn_b; nxt_q = nn_q;
  }
}

}  // namespace rfim
