// fd_u8_quad.cuh -- frequency-domain sigma cut (FDSC, Fig. 3) for uint8 dynamic spectra, one bin:
// the streaming kernel with one warp per 16-byte alignment class.
//
// Same idea as fd_u8_stream.cuh -- a tile (ALL channels x 128 samples of one beam) is streamed ONCE through small
// per-warp rings of TMA boxes, only exact column sums and one max / min SUMMARY per 4-channel x 4-sample block are
// kept, a threshold iteration is a packed test of the summaries plus an exact repair of the few candidate blocks
// through L1 / L2 -- with a different division of labour, chosen after the ncu capture of that kernel
// (profiles/r2a_*): a third of its warp time was spent at CTA-wide barriers of 16 warps and in repair loops whose
// trip count is the LARGEST candidate count among the 32 lanes of a warp (a lane owned 24 blocks, about one
// candidate each at k = 3, so three lanes in four idled through every trip).  Here
//   * a CTA is FOUR warps, warp w = alignment class w (rows w, w+4, ... of the beam: 4 * pitch bytes apart, a
//     multiple of 16, so one 2-D tensor map per class describes them even on the dense 12500-byte pitch); the four
//     warps are the whole barrier domain, every thread owns one of the 128 columns for the bounds (F3), and four or
//     five CTAs per SM fill each other's gaps;
//   * a lane sees C / 16 blocks, whose summaries live in shared memory (C / 8 bytes per lane);
//   * the candidates of a warp are POOLED: every lane appends its candidate blocks to a list in shared memory, and
//     the list is worked off 32 entries at a time, one block (4 rows x 4 bytes) per lane, with the column sums
//     corrected through shared-memory reductions.  A repair round now has 32 busy lanes.
// In place nothing but the replaced samples is written; out of place every word is copied in the statistics pass.
#pragma once

#include <cuda.h>

#include "common.cuh"
#include "packed.cuh"
#include "fd_u8_stream.cuh"   // FdStreamMaps / FdStreamParams, box geometry, fs_* helpers

namespace rfim {

constexpr int kFqWarps = 4;
constexpr int kFqThreads = 32 * kFqWarps;
constexpr int kFqMaxRing = 4;                        // boxes per warp ring (3 and 5 measured slower)
constexpr int kFqAhead = 0;                          // L2 prefetch distance in boxes; 0 = off (12 measured: 4.23 vs 3.63 ms)
constexpr int kFqDepth = 4;                          // repair rounds whose loads are in flight
constexpr int kFqListCap = 256;                      // candidate blocks per warp and repair chunk

struct __align__(16) FqCtrl {
  uint32_t acc[2][2 * kFsCols];                      // [buffer][S of 128 columns | Q of 128 columns]
  uint8_t lo[kFsCols], hi[kFsCols], rr[kFsCols];
  uint64_t full[kFqWarps][kFqMaxRing];               // ring mbarriers
  int tk[3][4];                                      // tile tickets handed to this CTA: {tile, beam, tile in beam}
  uint16_t list[kFqWarps][kFqListCap];               // candidate blocks of a warp: block << 5 | lane
};
// shared memory of one CTA: [rings: 4 warps x `ring` boxes][summaries: 4 warps x NBQ x 32 lanes x 16 bytes][FqCtrl]
__host__ __device__ inline size_t fd_quad_smem_bytes(int nbq, int ring) {
  return (size_t)kFqWarps * ring * kFsBoxWords * 4 + (size_t)kFqWarps * nbq * 32 * 16 + sizeof(FqCtrl);
}

// NBQ = boxes per warp and tile / 4 (C = 128 NBQ channels); kCopy: out of place; kRing: boxes per warp ring
template <int NBQ, bool kCopy, int kRing>
__global__ void __launch_bounds__(kFqThreads, kRing == 3 ? 5 : 4) fd_u8_quad_kernel(const __grid_constant__ FdStreamMaps maps,
                                                                   const FdStreamParams P) {
  extern __shared__ __align__(128) uint8_t smem[];
  constexpr int NB = 4 * NBQ;                        // boxes of 8 class rows per warp and tile
  constexpr int NW = (NBQ + 3) / 4;                  // 32-bit words of candidate bits per lane (8 bits per 4 boxes)
  const int tid = threadIdx.x, lane = tid & 31, cls = tid >> 5;
  const int C = P.C;
  constexpr int kFqSlots = kRing;
  uint32_t* const ring = reinterpret_cast<uint32_t*>(smem) + (size_t)cls * kFqSlots * kFsBoxWords;
  uint4* const sum4 = reinterpret_cast<uint4*>(smem + (size_t)kFqWarps * kFqSlots * kFsBoxWords * 4) + (size_t)cls * NBQ * 32;
  FqCtrl* const K = reinterpret_cast<FqCtrl*>(smem + (size_t)kFqWarps * kFqSlots * kFsBoxWords * 4 +
                                              (size_t)kFqWarps * NBQ * 32 * 16);
  uint64_t* const full = &K->full[cls][0];
  uint16_t* const list = &K->list[cls][0];

  if (tid == 0) {
#pragma unroll
    for (int k = 0; k < 4; ++k) fs_prefetch_desc(&maps.src[k]);
  }
  if (lane == 0) {
#pragma unroll
    for (int s = 0; s < kFqSlots; ++s) mbar_init(&full[s], 1);
    fence_mbar_init();
  }
  for (int i = tid; i < 4 * kFsCols; i += kFqThreads) (&K->acc[0][0])[i] = 0;

  // tiles are handed out by a ticket counter, in order, two tickets ahead (see fd_u8_stream.cuh)
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
  const int cq = C >> 2;                              // class rows per beam
  // box `c` of a tile: class rows [8 c, 8 c + 8) of the tile's beam, x = the tile's first column
  // bring a later box into L2 only: the ring holds kRing boxes per warp, DRAM latency under load is longer than
  // the time a warp takes to consume them, so the box kFqAhead boxes further on is requested early (no destination,
  // nothing to wait for) and its ring copy then comes out of L2
  auto prefetch = [&](int s0, int y0, int c) {        // one lane
    asm volatile("cp.async.bulk.prefetch.tensor.2d.L2.global.tile [%0, {%1, %2}];" ::"l"(
                     reinterpret_cast<uint64_t>(&maps.src[cls])),
                 "r"(s0), "r"(y0 + kFsBoxRows * c)
                 : "memory");
  };
  auto issue = [&](int s0, int y0, int c, int slot) {   // one lane
    mbar_arrive_expect_tx(&full[slot], kFsBoxWords * 4u);
    fs_tma_load_2d(ring + slot * kFsBoxWords, &maps.src[cls], s0, y0 + kFsBoxRows * c, &full[slot]);
  };
  if (lane == 0 && cur_t < P.total_tiles) {
#pragma unroll
    for (int c = 0; c < kFqSlots; ++c) issue(cur_q * kFsCols, (P.beam0 + cur_b) * cq, c, c);
  }

  uint32_t phases = 0;                                // one parity bit per ring slot
  int slot = 0;                                       // ring slot of the next box (boxes follow one another across tiles)
  int buf = 0;                                        // accumulator buffer of the next exchange
  uint32_t colS = 0, colQ = 0;                        // thread = column: exact totals, kept across iterations
  const int offw = P.off[cls] >> 2;                   // word offset of column s0 inside a box row
  const uint32_t* const lo32 = reinterpret_cast<const uint32_t*>(K->lo);
  const uint32_t* const hi32 = reinterpret_cast<const uint32_t*>(K->hi);
  const uint32_t* const rr32 = reinterpret_cast<const uint32_t*>(K->rr);

  while (cur_t < P.total_tiles) {
    const int b = P.beam0 + cur_b;
    const int s0 = cur_q * kFsCols;
    const bool have_next = nxt_t < P.total_tiles;
    const int nxt_s0 = nxt_q * kFsCols, nxt_y0 = (P.beam0 + nxt_b) * cq, cur_y0 = b * cq;
    const int tw = min(kFsCols, P.S - s0);            // valid columns of this tile
    const int nvalid = tw - 4 * lane;                 // valid bytes of this lane's word (>= 4: all)
    // class row j of this warp is channel 4 j + cls; consecutive class rows are 4 channels apart
    uint8_t* const dcls = P.dst + ((int64_t)b * C + cls) * P.stride + s0;
    const int64_t rstep = 4 * P.stride;

    // ------------------------------------------------------------------ F1 + F2: stream the rows once
    uint32_t S4[4] = {0, 0, 0, 0}, Q4[4] = {0, 0, 0, 0};
#pragma unroll 1
    for (int q = 0; q < NBQ; ++q) {
      uint32_t mx0 = 0, mx1 = 0, mn0 = 0, mn1 = 0;    // summaries of the 8 blocks of these 4 boxes
#pragma unroll
      for (int u = 0; u < 4; ++u) {                   // box c = 4 q + u lives in ring slot `slot`
        const int c = 4 * q + u;
        mbar_wait(&full[slot], (phases >> slot) & 1u);
        phases ^= 1u << slot;
        const uint32_t* rowp = ring + slot * kFsBoxWords + offw + lane;
        uint32_t w[kFsBoxRows];
#pragma unroll
        for (int j = 0; j < kFsBoxRows; ++j) w[j] = rowp[j * kFsPitchW];
        if (kCopy) {
          uint8_t* gd = dcls + (int64_t)(kFsBoxRows * c) * rstep + 4 * lane;
          if (nvalid >= 4) {
#pragma unroll
            for (int j = 0; j < kFsBoxRows; ++j) *reinterpret_cast<uint32_t*>(gd + j * rstep) = w[j];
          } else if (nvalid > 0) {
            for (int j = 0; j < kFsBoxRows; ++j)
              for (int v = 0; v < nvalid; ++v) gd[j * rstep + v] = (uint8_t)(w[j] >> (8 * v));
          }
        }
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          const uint32_t a = w[4 * h], bb = w[4 * h + 1], cc = w[4 * h + 2], d = w[4 * h + 3];
          const uint32_t ab_lo = prmt_b32(a, bb, 0x5140u), ab_hi = prmt_b32(a, bb, 0x7362u);
          const uint32_t cd_lo = prmt_b32(cc, d, 0x5140u), cd_hi = prmt_b32(cc, d, 0x7362u);
          const uint32_t t0 = prmt_b32(ab_lo, cd_lo, 0x5410u), t1 = prmt_b32(ab_lo, cd_lo, 0x7632u);
          const uint32_t t2 = prmt_b32(ab_hi, cd_hi, 0x5410u), t3 = prmt_b32(ab_hi, cd_hi, 0x7632u);
          S4[0] = __dp4a(t0, 0x01010101u, S4[0]); S4[1] = __dp4a(t1, 0x01010101u, S4[1]);
          S4[2] = __dp4a(t2, 0x01010101u, S4[2]); S4[3] = __dp4a(t3, 0x01010101u, S4[3]);
          Q4[0] = __dp4a(t0, t0, Q4[0]); Q4[1] = __dp4a(t1, t1, Q4[1]);
          Q4[2] = __dp4a(t2, t2, Q4[2]); Q4[3] = __dp4a(t3, t3, Q4[3]);
          const uint32_t e = group_summary(make_uint4(a, bb, cc, d));     // byte 1 = max, byte 0 = min
          constexpr uint32_t selx[4] = {0x3215u, 0x3250u, 0x3510u, 0x5210u};
          constexpr uint32_t seln[4] = {0x3214u, 0x3240u, 0x3410u, 0x4210u};
          const int blk = 2 * u + h;                  // block of this quartet of boxes: 0..7
          if (blk < 4) { mx0 = prmt(mx0, e, selx[blk & 3]); mn0 = prmt(mn0, e, seln[blk & 3]); }
          else         { mx1 = prmt(mx1, e, selx[blk & 3]); mn1 = prmt(mn1, e, seln[blk & 3]); }
        }
        // Refill the box only now: the statistics above have CONSUMED the eight words, so every lane's shared-memory
        // loads have completed (re-arming earlier lets the asynchronous copy overtake them).
        __syncwarp();
        if (lane == 0) {
          if (c + kFqSlots < NB) issue(s0, cur_y0, c + kFqSlots, slot);
          else if (have_next) issue(nxt_s0, nxt_y0, c + kFqSlots - NB, slot);
          if (kFqAhead > 0) {
            if (c + kFqAhead < NB) prefetch(s0, cur_y0, c + kFqAhead);
            else if (have_next) prefetch(nxt_s0, nxt_y0, c + kFqAhead - NB);
          }
        }
        slot = (slot + 1 == kFqSlots) ? 0 : slot + 1;
      }
      sum4[q * 32 + lane] = make_uint4(mx0, mx1, mn0, mn1);
    }
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      fs_red_add(&K->acc[buf][4 * lane + u], S4[u]);
      fs_red_add(&K->acc[buf][kFsCols + 4 * lane + u], Q4[u]);
    }

    // ------------------------------------------------------------------ F3..F5: thresholds
    int64_t nn_t = 0x7fffffff;
    int nn_b = 0, nn_q = 0;
    for (int it = 0; it < P.n_thr; ++it) {
      const bool first = it == 0;
      const bool need_stats = it + 1 < P.n_thr;
      // ---- exchange: accumulators -> column owners -> bounds for everybody
      __syncthreads();                                                // A: accumulators complete, repairs visible
      if (first && tid == kFqThreads - 1) take_ticket(2);             // the tile after the next one
      {
        const uint32_t s = K->acc[buf][tid], q = K->acc[buf][kFsCols + tid];
        if (first) { colS = s; colQ = q; } else { colS += s; colQ += q; }   // deltas are modulo 2^32
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
      }
      __syncthreads();                                                // B: bounds published
      if (first) { nn_t = K->tk[2][0]; nn_b = K->tk[2][1]; nn_q = K->tk[2][2]; }
      K->acc[buf][tid] = 0;                                           // nobody reads this buffer any more
      K->acc[buf][kFsCols + tid] = 0;
      buf ^= 1;

      // ---- candidate blocks of this lane from its summaries: bit (8 q + j) of hm <=> block j of box quartet q
      uint32_t hm[NW];
#pragma unroll
      for (int i = 0; i < NW; ++i) hm[i] = 0;
      {
        const uint32_t lo4 = lo32[lane], hi4 = hi32[lane];
        const uint32_t cab2 = (0x7fffu - fs_min4(hi4)) * 0x00010001u;
        const uint32_t cbe2 = (0x7fffu + fs_max4(lo4)) * 0x00010001u;
        if (nvalid > 0) {
#pragma unroll
          for (int q = 0; q < NBQ; ++q) {
            const uint4 s = sum4[q * 32 + lane];
            const uint32_t ma = bytes_above(s.x, cab2) | bytes_below(s.z, cbe2);
            const uint32_t mb = bytes_above(s.y, cab2) | bytes_below(s.w, cbe2);
            const uint32_t h8 = (((ma & 0x01010101u) * 0x01020408u) >> 24) | ((((mb & 0x01010101u) * 0x01020408u) >> 24) << 4);
            hm[q >> 2] |= h8 << (8 * (q & 3));
          }
        }
      }
      int mine = 0;
#pragma unroll
      for (int i = 0; i < NW; ++i) mine += __popc(hm[i]);

      // ---- pooled exact repair, through global memory (L1 / L2): chunks of at most kFqListCap blocks per warp
      uint32_t cnt_total = 0;
      while (true) {
        int incl = mine;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
          const int t = __shfl_up_sync(FULL, incl, o);
          if (lane >= o) incl += t;
        }
        const int total = __shfl_sync(FULL, incl, 31);
        if (total == 0) break;
        int pos = incl - mine;
        int room = max(0, kFqListCap - pos);                          // entries this lane may still append
#pragma unroll
        for (int i = 0; i < NW; ++i) {                                // one short loop per word of candidate bits
          while (hm[i] != 0u && room > 0) {
            const int bit = __ffs(hm[i]) - 1;
            hm[i] &= hm[i] - 1u;
            list[pos++] = (uint16_t)(((32 * i + bit) << 5) | lane);
            --room; --mine;
          }
        }
        __syncwarp();
        const int n = min(total, kFqListCap);
        // one entry = one block: 4 class rows x the 4 bytes of word column L.  The words of the next kFqDepth rounds are
        // requested before this round's are examined, so a round costs its instructions, not an L2 round trip.
        auto fetch = [&](int e, uint32_t& ent, uint32_t (&w4)[4]) {
          if (e < n) {
            ent = list[e];
            const int nvL = tw - 4 * (int)(ent & 31u);
            const uint8_t* gp = dcls + (int64_t)(4 * (int)(ent >> 5)) * rstep + 4 * (int)(ent & 31u);
            if (nvL >= 4) {
#pragma unroll
              for (int i = 0; i < 4; ++i) w4[i] = *reinterpret_cast<const uint32_t*>(gp + i * rstep);
            } else {
#pragma unroll
              for (int i = 0; i < 4; ++i) {
                w4[i] = 0;
                for (int v = 0; v < nvL; ++v) w4[i] |= (uint32_t)gp[i * rstep + v] << (8 * v);
              }
            }
          }
        };
        uint32_t ents[kFqDepth], ws[kFqDepth][4];
#pragma unroll
        for (int d = 0; d < kFqDepth; ++d) {
          ents[d] = 0;
#pragma unroll
          for (int i = 0; i < 4; ++i) ws[d][i] = 0;
          fetch(32 * d + lane, ents[d], ws[d]);
        }
        for (int e0 = 0; e0 < n; e0 += 32) {
          const bool have = e0 + lane < n;
          const uint32_t cent = ents[0];
          const uint32_t c0 = ws[0][0], c1 = ws[0][1], c2 = ws[0][2], c3 = ws[0][3];
#pragma unroll
          for (int d = 0; d + 1 < kFqDepth; ++d) {
            ents[d] = ents[d + 1];
#pragma unroll
            for (int i = 0; i < 4; ++i) ws[d][i] = ws[d + 1][i];
          }
          fetch(e0 + 32 * kFqDepth + lane, ents[kFqDepth - 1], ws[kFqDepth - 1]);
          if (have) {
            const int L = (int)(cent & 31u), blk = (int)(cent >> 5);
            const int nv = tw - 4 * L;                                // valid bytes of that word column
            const uint32_t lo4 = lo32[L], hi4 = hi32[L], r4 = rr32[L];
            const uint32_t chiE = 0x7fff7fffu - prmt_b32(hi4, 0u, 0x4240u), cloE = 0x80008000u - prmt_b32(lo4, 0u, 0x4240u);
            const uint32_t chiO = 0x7fff7fffu - prmt_b32(hi4, 0u, 0x4341u), cloO = 0x80008000u - prmt_b32(lo4, 0u, 0x4341u);
            uint32_t m0 = bytes_outside_cols(c0, chiE, cloE, chiO, cloO), m1 = bytes_outside_cols(c1, chiE, cloE, chiO, cloO);
            uint32_t m2 = bytes_outside_cols(c2, chiE, cloE, chiO, cloO), m3 = bytes_outside_cols(c3, chiE, cloE, chiO, cloO);
            if (nv < 4) {
              const uint32_t vm = (1u << (8 * nv)) - 1u;
              m0 &= vm; m1 &= vm; m2 &= vm; m3 &= vm;
            }
            if ((m0 | m1 | m2 | m3) != 0u) {
              uint8_t* const gp = dcls + (int64_t)(4 * blk) * rstep + 4 * L;
              const uint32_t n0 = (c0 & ~m0) | (r4 & m0), n1 = (c1 & ~m1) | (r4 & m1);
              const uint32_t n2 = (c2 & ~m2) | (r4 & m2), n3 = (c3 & ~m3) | (r4 & m3);
              if (nv >= 4) {
                if (m0) *reinterpret_cast<uint32_t*>(gp) = n0;
                if (m1) *reinterpret_cast<uint32_t*>(gp + rstep) = n1;
                if (m2) *reinterpret_cast<uint32_t*>(gp + 2 * rstep) = n2;
                if (m3) *reinterpret_cast<uint32_t*>(gp + 3 * rstep) = n3;
              } else {
                const uint32_t nn[4] = {n0, n1, n2, n3}, mm[4] = {m0, m1, m2, m3};
                for (int i = 0; i < 4; ++i)
                  for (int v = 0; v < nv; ++v)
                    if ((mm[i] >> (8 * v)) & 1u) gp[i * rstep + v] = (uint8_t)(nn[i] >> (8 * v));
              }
              if (P.flags) {
                const uint32_t mm[4] = {m0, m1, m2, m3};
                for (int i = 0; i < 4; ++i) {
                  uint8_t* fl = P.flags + ((int64_t)b * C + 4 * (4 * blk + i) + cls) * P.S + s0 + 4 * L;
#pragma unroll
                  for (int v = 0; v < 4; ++v)
                    if ((mm[i] >> (8 * v)) & 1u) fl[v] = 1;
                }
              }
              // per-column counts (one byte each) and, for the next iteration, the column deltas and a fresh summary
              const uint32_t cnt4 = (m0 & 0x01010101u) + (m1 & 0x01010101u) + (m2 & 0x01010101u) + (m3 & 0x01010101u);
              cnt_total += __dp4a(cnt4, 0x01010101u, 0u);
              if (need_stats) {
                // the replaced bytes, transposed: word u = the four rows of column u
                const uint32_t f0 = c0 & m0, f1 = c1 & m1, f2 = c2 & m2, f3 = c3 & m3;
                const uint32_t ab_lo = prmt_b32(f0, f1, 0x5140u), ab_hi = prmt_b32(f0, f1, 0x7362u);
                const uint32_t cd_lo = prmt_b32(f2, f3, 0x5140u), cd_hi = prmt_b32(f2, f3, 0x7362u);
                const uint32_t t[4] = {prmt_b32(ab_lo, cd_lo, 0x5410u), prmt_b32(ab_lo, cd_lo, 0x7632u),
                                       prmt_b32(ab_hi, cd_hi, 0x5410u), prmt_b32(ab_hi, cd_hi, 0x7632u)};
#pragma unroll
                for (int v = 0; v < 4; ++v) {
                  const uint32_t c = (cnt4 >> (8 * v)) & 0xffu;
                  if (c) {                                            // modulo 2^32: the column totals stay below 2^32
                    const uint32_t r = (r4 >> (8 * v)) & 0xffu;
                    fs_red_add(&K->acc[buf][4 * L + v], c * r - __dp4a(t[v], 0x01010101u, 0u));
                    fs_red_add(&K->acc[buf][kFsCols + 4 * L + v], c * r * r - __dp4a(t[v], t[v], 0u));
                  }
                }
                // the owner lane should not see this block as a candidate again for what has just been replaced
                const uint32_t e = group_summary(make_uint4(n0, n1, n2, n3));   // byte 1 = max, byte 0 = min
                uint8_t* sb = reinterpret_cast<uint8_t*>(&sum4[(blk >> 3) * 32 + L]) + ((blk >> 2) & 1) * 4 + (blk & 3);
                sb[0] = (uint8_t)(e >> 8);
                sb[8] = (uint8_t)e;
              }
            }
          }
        }
        __syncwarp();                                                 // the list is free for the next chunk
      }
      if (P.counts) {
        cnt_total = __reduce_add_sync(FULL, cnt_total);
        if (lane == 0 && cnt_total) atomicAdd(&P.counts[it], (unsigned long long)cnt_total);
      }
    }
    cur_t = nxt_t; cur_b = nxt_b; cur_q = nxt_q;
    nxt_t = nn_t; nxt_b = nn_b; nxt_q = nn_q;
  }
}

}  // namespace rfim
