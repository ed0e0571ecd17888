// fd_u8_qbin.cuh -- frequency-domain sigma cut (FDSC, Fig. 3) for uint8 dynamic spectra WITH the
// paper's per-bin mean correction (PAPER.md:102 step 1, :126): one streaming pass per step.
//
// Why not the summaries of fd_u8_stream.cuh / fd_u8_quad.cuh.  Those kernels stream a tile once, keep one max / min
// summary per 4 x 4 block and repair the few candidate blocks through L1 / L2.  At the paper's FDSC setting (bins of
// 32 channels, 2.75 sigma) candidates are not few: the kept interval differs from bin to bin AND from
// column to column (a bin mean of 32 samples is noisy), so one block in six is a candidate in the first iteration and
// one in ten in the second.  The ncu captures (profiles/r2i_*) show what that costs: 88 % of the instructions of the
// binned stream kernel are repair; with the repair pooled per warp (the quad kernel's scheme) the instruction count
// halves but the time does not (2.68 -> 2.46 ms on 96 beams), because every candidate is a gather of four 32-byte
// sectors of which 70 % miss L2 by the time the tile has been streamed (20 sectors per request, 1.6 x the batch in
// DRAM reads, long / short scoreboard stalls on 50 % of the samples).
//
// So this kernel reads a tile (ALL channels x 128 samples of one beam) 1 + n_thresholds times, every time as a stream
// of TMA boxes through the per-warp rings, which costs bandwidth the path has to spare instead of latency it has not:
//   pass 0          column totals Q and per (bin, column) sums S_b (two 16-bit fields per word, RED.ADD from all
//                   warps); out of place it also copies every word to the destination;
//   F3, per step    one thread per column: V = nb Q - sum_b S_b^2, T = isqrt(floor(p^2 nb V / (2^32 C))); then all
//                   threads: lo = ceil((S_b - T) / nb), hi = floor((S_b + T) / nb), r = rounded S_b / nb for every
//                   (bin, column), four columns per thread;
//   pass 1 + i      iteration i over the DESTINATION (its own tensor maps): exact per-byte masks against the bounds
//                   of the block's bin, replaced words stored (nothing else is written), and Q and S_b of the data as
//                   it now stands for the next step.  Branch-free: at 2.75 sigma some lane of a warp has a hit in
//                   every block.
// A CTA is eight warps (alignment class x half of the channels, as many barrier domains as SMs x 3); the rings run
// across passes and tiles (the first boxes of the next pass are requested while this one ends -- a warp only ever
// re-reads what it wrote itself, ordered by a proxy fence).  Integer arithmetic is the oracle's
// (flag <=> (nb x - S_b)^2 > floor(p^2 nb V / (2^32 C))): bit-exact.
#pragma once

#include <cuda.h>

#include "common.cuh"
#include "packed.cuh"
#include "fd_u8_stream.cuh"   // FdStreamParams, box geometry, fs_* helpers

namespace rfim {

constexpr int kQbWarps = 8;                          // warp = (alignment class, half of the channels)
constexpr int kQbThreads = 32 * kQbWarps;
constexpr int kQbRing = 4;                           // boxes per warp ring

struct FdQbMaps {
  CUtensorMap src[4];                                // one per alignment class (row mod 4)
  CUtensorMap dst[4];                                // the same for the destination (in place: equal to src)
};

struct __align__(16) QbCtrl {
  uint32_t acc[kFsCols];                             // Q of 128 columns, summed by the pass before a step
  uint32_t T[kFsCols];                               // per-column threshold on |nb x - S_b|
  uint64_t full[kQbWarps][kQbRing];                  // ring mbarriers
  int tk[3][4];                                      // tile tickets handed to this CTA: {tile, beam, tile in beam}
};
// shared memory of one CTA: [rings: 8 warps x 4 boxes][QbCtrl][binS[nbins][64] u32][lo, hi, r [nbins][128] u8]
__host__ __device__ inline size_t fd_qbin_smem_bytes(int nbins) {
  return (size_t)kQbWarps * kQbRing * kFsBoxWords * 4 + sizeof(QbCtrl) + (size_t)nbins * (kFsCols / 2) * 4 +
         (size_t)3 * nbins * kFsCols;
}

__device__ __forceinline__ void fence_proxy_async_global() {
  asm volatile("fence.proxy.async.global;" ::: "memory");
}

// NB = boxes of 8 class rows per warp and tile (C = 64 NB channels); kCopy: out of place; kOut: flags or counts wanted
template <int NB, bool kCopy, bool kOut>
__global__ void __launch_bounds__(kQbThreads, 3) fd_u8_qbin_kernel(const __grid_constant__ FdQbMaps maps,
                                                                  const FdStreamParams P) {
  extern __shared__ __align__(128) uint8_t smem[];
  constexpr int RWC = kFsBoxRows * NB;               // class rows per warp
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int cls = warp & 3, g = warp >> 2;
  const int C = P.C, nbins = P.nbins;
  uint32_t* const ring = reinterpret_cast<uint32_t*>(smem) + (size_t)warp * kQbRing * kFsBoxWords;
  uint8_t* sp = smem + (size_t)kQbWarps * kQbRing * kFsBoxWords * 4;
  QbCtrl* const K = reinterpret_cast<QbCtrl*>(sp);
  sp += sizeof(QbCtrl);
  uint32_t* const bS = reinterpret_cast<uint32_t*>(sp);             // [nbins][64]: two columns per word
  sp += (size_t)nbins * (kFsCols / 2) * 4;
  uint32_t* const lo32 = reinterpret_cast<uint32_t*>(sp);           // [nbins][128] bytes each
  uint32_t* const hi32 = lo32 + nbins * (kFsCols / 4);
  uint32_t* const rr32 = hi32 + nbins * (kFsCols / 4);
  uint64_t* const full = &K->full[warp][0];

  if (tid == 0) {
#pragma unroll
    for (int k = 0; k < 4; ++k) { fs_prefetch_desc(&maps.src[k]); fs_prefetch_desc(&maps.dst[k]); }
  }
  if (lane == 0) {
#pragma unroll
    for (int s = 0; s < kQbRing; ++s) mbar_init(&full[s], 1);
    fence_mbar_init();
  }
  for (int i = tid; i < kFsCols; i += kQbThreads) K->acc[i] = 0;
  for (int i = tid; i < nbins * (kFsCols / 2); i += kQbThreads) bS[i] = 0;

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
  const int ywarp = g * RWC;                          // the warp's first class row inside a beam
  // box `c` of a pass: class rows [8 c, 8 c + 8) of the warp, of the source (pass 0) or the destination
  auto issue = [&](const CUtensorMap* map, int s0, int y0, int c, int slot) {   // one lane
    mbar_arrive_expect_tx(&full[slot], kFsBoxWords * 4u);
    fs_tma_load_2d(ring + slot * kFsBoxWords, map, s0, y0 + kFsBoxRows * c, &full[slot]);
  };
  if (lane == 0 && cur_t < P.total_tiles) {
#pragma unroll
    for (int c = 0; c < kQbRing; ++c) issue(&maps.src[cls], cur_q * kFsCols, (P.beam0 + cur_b) * cq + ywarp, c, c);
  }

  // a block is 4 class rows = 16 consecutive channels; a bin is bpb whole blocks and does not straddle warps (host)
  const int bpb = P.nb >> 4;
  const int bin0 = (4 * ywarp) / P.nb;                // bin of the warp's block 0

  uint32_t phases = 0;                                // one parity bit per ring slot
  int slot = 0;                                       // ring slot of the next box (boxes follow one another)
  const int offs = P.off[cls] >> 2, offd = P.off_dst[cls] >> 2;   // word offset of column s0 inside a box row

  while (cur_t < P.total_tiles) {
    const int b = P.beam0 + cur_b;
    const int s0 = cur_q * kFsCols;
    const bool have_next = nxt_t < P.total_tiles;
    const int nxt_s0 = nxt_q * kFsCols, nxt_y0 = (P.beam0 + nxt_b) * cq + ywarp, cur_y0 = b * cq + ywarp;
    const int tw = min(kFsCols, P.S - s0);            // valid columns of this tile
    const int nvalid = tw - 4 * lane;                 // valid bytes of this lane's word (>= 4: all)
    // class row j of this warp is channel 4 (ywarp + j) + cls; consecutive class rows are 4 channels apart
    uint8_t* const dcls = P.dst + ((int64_t)b * C + 4 * ywarp + cls) * P.stride + s0 + 4 * lane;
    const int64_t rstep = 4 * P.stride;
    // the box that takes the place of box c of pass `pass` in the ring: box c + 4 of the same pass, or of the next
    // pass over this tile (always the destination), or of pass 0 of the next tile
    auto refill = [&](int pass, int c) {              // one lane
      if (c + kQbRing < NB) issue(pass == 0 ? &maps.src[cls] : &maps.dst[cls], s0, cur_y0, c + kQbRing, slot);
      else if (pass < P.n_thr) issue(&maps.dst[cls], s0, cur_y0, c + kQbRing - NB, slot);
      else if (have_next) issue(&maps.src[cls], nxt_s0, nxt_y0, c + kQbRing - NB, slot);
    };

    // ------------------------------------------------------------------ pass 0 (F1 + F2): totals and bin sums
    {
      uint32_t Q4[4] = {0, 0, 0, 0};
      uint32_t B4[4] = {0, 0, 0, 0};                  // sums of the bin being streamed
      int fbin = bin0, left = bpb;                    // that bin, and the blocks it still lacks
#pragma unroll 2
      for (int c = 0; c < NB; ++c) {
        mbar_wait(&full[slot], (phases >> slot) & 1u);
        phases ^= 1u << slot;
        const uint32_t* rowp = ring + slot * kFsBoxWords + offs + lane;
        uint32_t w[kFsBoxRows];
#pragma unroll
        for (int j = 0; j < kFsBoxRows; ++j) w[j] = rowp[j * kFsPitchW];
        if (kCopy) {
          uint8_t* gd = dcls + (int64_t)(kFsBoxRows * c) * rstep;
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
          B4[0] = __dp4a(t0, 0x01010101u, B4[0]); B4[1] = __dp4a(t1, 0x01010101u, B4[1]);
          B4[2] = __dp4a(t2, 0x01010101u, B4[2]); B4[3] = __dp4a(t3, 0x01010101u, B4[3]);
          Q4[0] = __dp4a(t0, t0, Q4[0]); Q4[1] = __dp4a(t1, t1, Q4[1]);
          Q4[2] = __dp4a(t2, t2, Q4[2]); Q4[3] = __dp4a(t3, t3, Q4[3]);
          if (--left == 0) {                          // warp-uniform: the bin ends with this block (S_b <= 255 nb < 2^16)
            fs_red_add(&bS[fbin * (kFsCols / 2) + 2 * lane], B4[0] | (B4[1] << 16));
            fs_red_add(&bS[fbin * (kFsCols / 2) + 2 * lane + 1], B4[2] | (B4[3] << 16));
            B4[0] = 0; B4[1] = 0; B4[2] = 0; B4[3] = 0;
            ++fbin;
            left = bpb;
          }
        }
        // Refill the box only now: the statistics above have CONSUMED the eight words, so every lane's shared-memory
        // loads have completed (re-arming earlier lets the asynchronous copy overtake them).  Out of place the next
        // pass reads what this warp has just copied: generic-proxy stores -> async-proxy loads need the fence.
        if (kCopy && c + kQbRing >= NB) fence_proxy_async_global();   // (every lane, after its own stores)
        __syncwarp();
        if (lane == 0) refill(0, c);
        slot = (slot + 1 == kQbRing) ? 0 : slot + 1;
      }
#pragma unroll
      for (int u = 0; u < 4; ++u) fs_red_add(&K->acc[4 * lane + u], Q4[u]);
    }

    // ------------------------------------------------------------------ F3..F5: one pass per threshold
    int64_t nn_t = 0x7fffffff;
    int nn_b = 0, nn_q = 0;
    for (int it = 0; it < P.n_thr; ++it) {
      const bool first = it == 0;
      const bool need_stats = it + 1 < P.n_thr;
      // ---- step 1: one thread per column, V = nb Q - sum_b S_b^2 and T = isqrt(floor(p^2 nb V / (2^32 C)))
      __syncthreads();                                                // A: Q and bin sums (or their deltas) complete
      if (first && tid == kQbThreads - 1) take_ticket(2);             // the tile after the next one
      if (tid < kFsCols) {
        const uint32_t colQ = K->acc[tid];                                           // the pass before this step left the totals
        K->acc[tid] = 0;                                              // read by this thread only
        uint64_t ss = 0;
        const int sh = (tid & 1) * 16;
        const uint32_t* bp = bS + (tid >> 1);
#pragma unroll 4
        for (int bn = 0; bn < nbins; ++bn) {
          const uint32_t sb = (bp[bn * (kFsCols / 2)] >> sh) & 0xffffu;
          ss += (uint64_t)sb * sb;
        }
        const uint64_t V = (uint64_t)P.nb * colQ - ss;
        const uint64_t nbV = (uint64_t)P.nb * V;                      // < 2^45 (nb <= 256, C <= 4096)
        const uint64_t p2 = (uint64_t)P.p[it] * P.p[it];
        const uint64_t xh = __umul64hi(p2, nbV), xl = p2 * nbV;       // p^2 nb V < 2^93
        const uint64_t Y = (xh << 32) | (xl >> 32);                   // floor(p^2 nb V / 2^32) < 2^61
        const uint64_t W = fs_div_u64(Y, (uint32_t)C);
        uint64_t T = (uint64_t)__dsqrt_rd((double)W);
        while (T * T > W) --T;
        while ((T + 1) * (T + 1) <= W) ++T;
        K->T[tid] = tid < tw ? (uint32_t)min(T, (uint64_t)0xffffu) : 0xffffu;   // |nb x - S_b| <= 255 nb < 65535
      }
      __syncthreads();                                                // A2: thresholds published
      // ---- step 2: (bin, word column) -> bounds of its four columns.
      // umulhi(a, ceil(2^32 / n)) = floor(a / n) exactly while a n < 2^32: here a < 2^18 and n <= 512.
      {
        const uint4 T4 = reinterpret_cast<const uint4*>(K->T)[lane];
        const uint32_t Tc[4] = {T4.x, T4.y, T4.z, T4.w};
        const uint32_t nb = (uint32_t)P.nb;
        for (int bn = warp; bn < nbins; bn += kQbWarps) {
          uint2* const sp2 = reinterpret_cast<uint2*>(bS) + bn * 32 + lane;
          const uint2 sb2 = *sp2;
          *sp2 = make_uint2(0u, 0u);                                  // the coming pass (or the next tile) sums afresh
          const uint32_t sbs[4] = {sb2.x & 0xffffu, sb2.x >> 16, sb2.y & 0xffffu, sb2.y >> 16};
          uint32_t lo4 = 0, hi4 = 0, r4 = 0;
#pragma unroll
          for (int v = 0; v < 4; ++v) {
            const uint32_t sb = sbs[v], T = Tc[v];
            uint32_t hi = min(__umulhi(sb + T, P.inv_nb), 255u);
            uint32_t lo = sb > T ? __umulhi(sb - T + nb - 1u, P.inv_nb) : 0u;
            if (lo > hi) { lo = 1; hi = 0; }
            const uint32_t r = __umulhi(2u * sb + nb, P.inv_2nb);
            lo4 |= lo << (8 * v); hi4 |= hi << (8 * v); r4 |= r << (8 * v);
          }
          lo32[bn * 32 + lane] = lo4;
          hi32[bn * 32 + lane] = hi4;
          rr32[bn * 32 + lane] = r4;
        }
      }
      __syncthreads();                                                // B: bounds published
      if (first) { nn_t = K->tk[2][0]; nn_b = K->tk[2][1]; nn_q = K->tk[2][2]; }

      // ---- pass 1 + it over the destination: exact masks, replace, and the sums of the replaced data for the next step
      uint32_t pc = 0;                                                // 8 x replaced bytes of this lane
      uint32_t Q4[4] = {0, 0, 0, 0}, B4[4] = {0, 0, 0, 0};
      uint32_t r4 = 0, chiE = 0, cloE = 0, chiO = 0, cloO = 0;        // bounds of the bin being streamed
      int fbin = bin0, left = bpb;
      bool fresh = true;
      // (bytes beyond the row end are zero-filled and their columns have T = 65535: lo = 0, hi = 255, never cut)
      const bool want_counts = kOut && P.counts != nullptr, want_flags = kOut && P.flags != nullptr;
      uint8_t* gp = dcls;                                             // first row of the coming block
#pragma unroll 1
      for (int c = 0; c < NB; ++c) {
        mbar_wait(&full[slot], (phases >> slot) & 1u);
        phases ^= 1u << slot;
        const uint32_t* rowp = ring + slot * kFsBoxWords + offd + lane;
        uint32_t w[kFsBoxRows];
#pragma unroll
        for (int j = 0; j < kFsBoxRows; ++j) w[j] = rowp[j * kFsPitchW];
#pragma unroll
        for (int h = 0; h < 2; ++h, gp += 4 * rstep) {
          if (fresh) {                                                // warp-uniform: a new bin starts with this block
            const uint32_t lo4 = lo32[fbin * 32 + lane], hi4 = hi32[fbin * 32 + lane];
            r4 = rr32[fbin * 32 + lane];
            chiE = 0x7fff7fffu - prmt_b32(hi4, 0u, 0x4240u); cloE = 0x80008000u - prmt_b32(lo4, 0u, 0x4240u);
            chiO = 0x7fff7fffu - prmt_b32(hi4, 0u, 0x4341u); cloO = 0x80008000u - prmt_b32(lo4, 0u, 0x4341u);
            fresh = false;
          }
          const uint32_t c0 = w[4 * h], c1 = w[4 * h + 1], c2 = w[4 * h + 2], c3 = w[4 * h + 3];
          const uint32_t m0 = bytes_outside_cols(c0, chiE, cloE, chiO, cloO);
          const uint32_t m1 = bytes_outside_cols(c1, chiE, cloE, chiO, cloO);
          const uint32_t m2 = bytes_outside_cols(c2, chiE, cloE, chiO, cloO);
          const uint32_t m3 = bytes_outside_cols(c3, chiE, cloE, chiO, cloO);
          const uint32_t n0 = (c0 & ~m0) | (r4 & m0), n1 = (c1 & ~m1) | (r4 & m1);
          const uint32_t n2 = (c2 & ~m2) | (r4 & m2), n3 = (c3 & ~m3) | (r4 & m3);
          if (nvalid >= 4) {
            if (m0) *reinterpret_cast<uint32_t*>(gp) = n0;
            if (m1) *reinterpret_cast<uint32_t*>(gp + rstep) = n1;
            if (m2) *reinterpret_cast<uint32_t*>(gp + 2 * rstep) = n2;
            if (m3) *reinterpret_cast<uint32_t*>(gp + 3 * rstep) = n3;
          } else if ((m0 | m1 | m2 | m3) != 0u) {
            const uint32_t nn[4] = {n0, n1, n2, n3}, mm[4] = {m0, m1, m2, m3};
            for (int i = 0; i < 4; ++i)
              for (int v = 0; v < nvalid; ++v)
                if ((mm[i] >> (8 * v)) & 1u) gp[i * rstep + v] = (uint8_t)(nn[i] >> (8 * v));
          }
          if (want_flags && (m0 | m1 | m2 | m3) != 0u) {
            const uint32_t mm[4] = {m0, m1, m2, m3};
            for (int i = 0; i < 4; ++i) {
              uint8_t* fl = P.flags + ((int64_t)b * C + 4 * (ywarp + kFsBoxRows * c + 4 * h + i) + cls) * P.S + s0 + 4 * lane;
#pragma unroll
              for (int v = 0; v < 4; ++v)
                if ((mm[i] >> (8 * v)) & 1u) fl[v] = 1;
            }
          }
          if (want_counts) pc += __popc(m0) + __popc(m1) + __popc(m2) + __popc(m3);
          if (need_stats) {
            // the next step's statistics are those of the data as it now stands: sum it as pass 0 did (cheaper
            // than deltas of the replaced bytes, which need their count per column on top)
            const uint32_t ab_lo = prmt_b32(n0, n1, 0x5140u), ab_hi = prmt_b32(n0, n1, 0x7362u);
            const uint32_t cd_lo = prmt_b32(n2, n3, 0x5140u), cd_hi = prmt_b32(n2, n3, 0x7362u);
            const uint32_t t0 = prmt_b32(ab_lo, cd_lo, 0x5410u), t1 = prmt_b32(ab_lo, cd_lo, 0x7632u);
            const uint32_t t2 = prmt_b32(ab_hi, cd_hi, 0x5410u), t3 = prmt_b32(ab_hi, cd_hi, 0x7632u);
            B4[0] = __dp4a(t0, 0x01010101u, B4[0]); B4[1] = __dp4a(t1, 0x01010101u, B4[1]);
            B4[2] = __dp4a(t2, 0x01010101u, B4[2]); B4[3] = __dp4a(t3, 0x01010101u, B4[3]);
            Q4[0] = __dp4a(t0, t0, Q4[0]); Q4[1] = __dp4a(t1, t1, Q4[1]);
            Q4[2] = __dp4a(t2, t2, Q4[2]); Q4[3] = __dp4a(t3, t3, Q4[3]);
          }
          if (--left == 0) {                                          // warp-uniform: the bin ends with this block
            if (need_stats) {
              fs_red_add(&bS[fbin * (kFsCols / 2) + 2 * lane], B4[0] | (B4[1] << 16));
              fs_red_add(&bS[fbin * (kFsCols / 2) + 2 * lane + 1], B4[2] | (B4[3] << 16));
              B4[0] = 0; B4[1] = 0; B4[2] = 0; B4[3] = 0;
            }
            ++fbin;
            left = bpb;
            fresh = true;
          }
        }
        // the next pass re-reads what this warp has stored: generic-proxy stores -> async-proxy loads (every lane
        // fences after its own stores; the boxes concerned were written at least NB - 4 boxes ago)
        if (c + kQbRing >= NB) fence_proxy_async_global();
        __syncwarp();
        if (lane == 0) refill(it + 1, c);
        slot = (slot + 1 == kQbRing) ? 0 : slot + 1;
      }
      if (need_stats) {
#pragma unroll
        for (int u = 0; u < 4; ++u) fs_red_add(&K->acc[4 * lane + u], Q4[u]);
      }
      if (want_counts) {
        const uint32_t cnt_total = __reduce_add_sync(FULL, pc >> 3);
        if (lane == 0 && cnt_total) atomicAdd(&P.counts[it], (unsigned long long)cnt_total);
      }
    }
    cur_t = nxt_t; cur_b = nxt_b; cur_q = nxt_q;
    nxt_t = nn_t; nxt_b = nn_b; nxt_q = nn_q;
  }
}

}  // namespace rfim
