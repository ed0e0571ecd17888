// fd_u8_strip.cuh -- frequency-domain sigma cut (FDSC, Fig. 3) for uint8 dynamic spectra,
// one bin of all channels: the strip kernel.
//
// The general fast kernel: any channel count that is a multiple of 4 (up to ~12 K channels through clusters of
// CTAs), mean replacement, or -- for tiles that fit one CTA -- the median (kMedian).  Auto mode takes it for short
// batches and out of place; large in-place batches go to the streaming kernel of fd_u8_quad.cuh, bins to
// fd_u8_stream.cuh (launch_fd_misc.cu has the order and the measurements behind it).
//
// A tile is ALL channels x 128 consecutive samples of one beam (a strip), resident in shared memory as rows of
// 144 bytes.  Whenever it fits (<= 1576 channels) ONE CTA of 32 warps holds the whole tile (216 KB, one CTA per
// SM, only __syncthreads); otherwise the channels are split over the smallest thread-block cluster that fits,
// CTA q holding channels [q*Rq, (q+1)*Rq), and column statistics / bounds cross the cluster through DSMEM.
//   F1: TMA tensor copies, one box per warp (or per alignment class): the rows of one 16-byte alignment class
//       (row mod 4) form a 2-D tensor even on the dense 4-byte aligned pitch; a box is the 144-byte aligned
//       superset of the 128 columns.  Fallback (channels % 4 != 0, variant 13): one 1-D bulk copy per row.
//   F2: lane = word column (32 lanes x 4 samples = the strip); a warp reads 32 consecutive words of one row (no
//       bank conflicts).  4x4 byte transposes (PRMT) turn four rows into words that each hold ONE column, so
//       IDP.4A gives exact column sums and sums of squares; the warps meet in shared-memory accumulators (RED.ADD).
//   F3: column c is owned by one thread of one CTA, which adds up the accumulators of all CTAs, keeps (S, Q) in
//       registers across iterations, computes the exact kept interval [lo, hi] in closed form (integer square
//       root) and r, and publishes them to every CTA.
//   F4: packed range check per four rows (VIADDMNMX.U16x2) records which steps hold an outlier; the exact
//       repair runs afterwards over the recorded steps only; column deltas go to the accumulators.
//   F5: next threshold from the updated (S, Q).  F6: out of place a full-width tile is copied to the destination
//       while F2 reads it, and from then on only repaired rows are written, as in place; otherwise the last sweep
//       writes the rows it finds clean straight from its registers, the repair writes the others.  Always one
//       coalesced 32-bit store per lane and row (the 144-byte
//       superset cannot be stored back by TMA: its margins belong to the neighbouring tiles, a tensor box must
//       start on a 16-byte boundary and TMA stores clip at 16-byte granularity).
#pragma once

#include <cuda.h>   // CUtensorMap (types only: the encoder is fetched through the runtime, no -lcuda)

#include "common.cuh"
#include "packed.cuh"

namespace rfim {

constexpr int kStripWords = 32;                  // word columns per tile (128 samples)
constexpr int kStripCols = 4 * kStripWords;
constexpr int kStripPitchW = 36;                 // bulk path: row pitch in words: 128 bytes + up to 12 bytes of phase + rounding

struct FdStripParams {
  const uint8_t* src;
  uint8_t* dst;
  int64_t stride;
  int beams, C, S;
  int n_thr;
  uint32_t p[16];
  uint8_t* flags;
  unsigned long long* counts;
  int Rq;                       // channels per CTA
  int tiles_per_beam;
  int64_t total_tiles;
  int off[4];                   // tensor path: x offset (bytes) of row class k inside its 16-byte aligned tensor
  int box_rows;                 // tensor path: rows per tensor copy (divides Rq / 4, <= 256)
  uint32_t invC;                // ceil(2^32 / C) for C >= 2 (32-bit quotients of the bounds), else 0
};

// Tensor path.  Issuing one bulk copy per 128-byte row segment costs about ten warp instructions per copy
// (the copy takes uniform operands, so a warp issues its lanes' copies one after the other): a third of the
// kernel's instructions.  Rows 4 apart are 4 * pitch bytes apart, a multiple of 16, so the rows of one
// 16-byte alignment class (row mod 4) form a 2-D tensor a TMA tensor map can describe: base rounded down to
// 16 bytes, x counted from there.  A box must start on a 16-byte boundary, so the box is the 144-byte aligned
// superset of the 128 columns (x = s0, the tile's first column sits off[k] bytes into the box) and one tensor
// copy moves a whole class of a CTA's rows (Rq / 4 <= 256 rows): four copies per CTA and tile; columns
// beyond the row end are zero-filled by the hardware.  The superset cannot be stored back (its margins
// belong to the neighbouring tiles), so F6 writes each 128-byte row segment with one coalesced 32-bit store
// per lane.
struct FdStripMaps {
  CUtensorMap src[4];
};
__device__ __forceinline__ void tma_load_2d(void* smem_dst, const CUtensorMap* map, int x, int y, uint64_t* bar) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
      ::"r"(smem_addr(smem_dst)), "l"(reinterpret_cast<uint64_t>(map)), "r"(x), "r"(y), "r"(smem_addr(bar))
      : "memory");
}
// bring a box into L2 only (no shared-memory destination, no completion to wait for)
__device__ __forceinline__ void tma_prefetch_l2_2d(const CUtensorMap* map, int x, int y) {
  asm volatile("cp.async.bulk.prefetch.tensor.2d.L2.global.tile [%0, {%1, %2}];" ::"l"(reinterpret_cast<uint64_t>(map)),
               "r"(x), "r"(y)
               : "memory");
}
__device__ __forceinline__ void tma_prefetch_desc(const CUtensorMap* map) {
  asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(map)) : "memory");
}

// control area behind the rows
struct __align__(16) FdStripCtrl {
  uint32_t acc[2][2 * kStripCols];               // [buffer][S of 128 columns, Q of 128 columns]
  uint4 chk[kStripWords];                        // per word column {negE, negO, thrE, thrO}
  uint8_t lo[kStripCols], hi[kStripCols], rr[kStripCols];
  uint64_t bar[32];                              // tensor path: one per alignment class, or one per warp (kWarpBox); bulk path: bar[0]
  uint32_t cnt[kStripCols];                      // kMedian: samples above the probe value, per column
  uint8_t mid[kStripCols];                       // kMedian: probe value of the bisection, per column
};
__host__ __device__ inline size_t fd_strip_smem_bytes(int Rq) {
  return (size_t)Rq * kStripPitchW * 4 + sizeof(FdStripCtrl);
}

__device__ __forceinline__ void dsmem_st_u8(uint32_t addr, uint32_t v) {
  asm volatile("st.shared::cluster.u8 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}
__device__ __forceinline__ void dsmem_st_u16(uint32_t addr, uint32_t v) {
  asm volatile("st.shared::cluster.u16 [%0], %1;" ::"r"(addr), "h"((unsigned short)v) : "memory");
}
__device__ __forceinline__ void smem_red_add(uint32_t* p, uint32_t v) {
  asm volatile("red.shared.add.u32 [%0], %1;" ::"r"(smem_addr(p)), "r"(v) : "memory");
}

// NW warps per CTA: 16 (two CTAs per SM) or 32 (one CTA per SM holding a whole tile).
// kWarpBox (tensor path, Rq a multiple of 8 NW): a warp owns Rq / NW CONSECUTIVE rows of its alignment class, one
// tensor box with its own mbarrier, so every warp runs its own copy-in / store / next-copy-in pipeline and no warp
// waits for the slowest warp of its class before the next tile's rows are requested.
// kMedian (single CTA per tile only): the replacement value is the column's lower median, found once
// per column on the resident tile by bisection over the byte values with packed counting passes.
template <bool kTensor, int NW, bool kWarpBox, bool kMedian = false>
__global__ void __launch_bounds__(32 * NW, NW == 16 ? 2 : 1) fd_u8_strip_kernel(const __grid_constant__ FdStripMaps maps,
                                                                                const FdStripParams P) {
  constexpr int kStripThreads = 32 * NW, kStripWarps = NW;
  extern __shared__ __align__(128) uint8_t smem[];
  constexpr int PW = kStripPitchW;
  // words between consecutive rows (16 apart) of one thread.  Tensor path: the rows of alignment class k are
  // stored together (class-major), local row r at shared-memory row (r & 3) * Rq / 4 + (r >> 2).
  constexpr int RS = kWarpBox ? PW : kTensor ? (NW / 4) * PW : kStripWarps * PW;
  const int C = P.C, Rq = P.Rq;
  uint32_t* tile = reinterpret_cast<uint32_t*>(smem);
  FdStripCtrl* K = reinterpret_cast<FdStripCtrl*>(smem + (size_t)Rq * PW * 4);
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const uint32_t rank = cluster_ctarank(), ncta = cluster_nctarank();
  const int c0 = (int)rank * Rq;                      // first channel of this CTA
  const int nrows = max(0, min(Rq, C - c0));
  const int ni = kWarpBox ? Rq / NW : nrows > warp ? (nrows - warp + kStripWarps - 1) / kStripWarps : 0;   // rows of this thread
  // logical row (channel - c0) of this thread's i-th row: row0 + rowmul * i
  const int row0 = kWarpBox ? 4 * ((warp >> 2) * ni) + (warp & 3) : warp;
  constexpr int rowmul = kWarpBox ? 4 : kStripWarps;
  const int cpc = kStripCols / (int)ncta;             // columns owned per CTA (F3)
  const bool owner = tid < cpc;
  const int ocol = (int)rank * cpc + tid;
  const int nload = min(nrows, kStripThreads);
  auto sync_all = [&]() { if (ncta > 1) cluster_sync_all(); else __syncthreads(); };

  if (tid == 0) {
    if (kTensor) {
#pragma unroll
      for (int k = 0; k < (kWarpBox ? NW : 4); ++k) mbar_init(&K->bar[k], 1);
    } else {
      mbar_init(&K->bar[0], nload > 0 ? nload : 1);
    }
    fence_mbar_init();
    if (kTensor) {
#pragma unroll
      for (int k = 0; k < 4; ++k) tma_prefetch_desc(&maps.src[k]);
    }
  }
  for (int i = tid; i < 4 * kStripCols; i += kStripThreads) (&K->acc[0][0])[i] = 0;   // 2 x 256 accumulators
  __syncthreads();
  if (ncta > 1) cluster_sync_all();                   // peers' shared memory is live before any DSMEM access

  // Tensor path: the warps of one alignment class (warp & 3) depend only on that class's copies.  The loads of
  // class k of the NEXT tile are issued as soon as the class's warps have written their rows of this tile, so
  // they overlap the stores and the other classes' last sweep; statistics start per class as it arrives.
  const int cls = warp & 3;
  auto issue_class_load = [&](int64_t t, int k) {     // one thread
    const int b = (int)(t / P.tiles_per_beam);
    const int s0 = (int)(t % P.tiles_per_beam) * kStripCols;
    const int ycls = (int)(((int64_t)b * C + c0) >> 2);
    mbar_arrive_expect_tx(&K->bar[k], (uint32_t)(Rq >> 2) * PW * 4u);
    for (int y = 0; y < (Rq >> 2); y += P.box_rows)
      tma_load_2d(tile + ((size_t)k * (Rq >> 2) + y) * PW, &maps.src[k], s0, ycls + y, &K->bar[k]);
  };
  auto issue_warp_load = [&](int64_t t) {             // lane 0 of every warp: the warp's own box
    const int b = (int)(t / P.tiles_per_beam);
    const int s0 = (int)(t % P.tiles_per_beam) * kStripCols;
    const int ycls = (int)(((int64_t)b * C + c0) >> 2);
    mbar_arrive_expect_tx(&K->bar[warp], (uint32_t)ni * PW * 4u);
    tma_load_2d(tile + ((size_t)cls * (Rq >> 2) + (size_t)(warp >> 2) * ni) * PW, &maps.src[cls], s0,
                ycls + (warp >> 2) * ni, &K->bar[warp]);
  };
  const uint32_t nclusters = cluster_nid_x();
  if (kWarpBox) {
    if (lane == 0 && (int64_t)cluster_id_x() < P.total_tiles) issue_warp_load(cluster_id_x());
  } else if (kTensor && tid < 4 && (int64_t)cluster_id_x() < P.total_tiles) {
    issue_class_load(cluster_id_x(), tid);
  }

  uint32_t phase = 0;
  int buf = 0;                                        // accumulator buffer of the next exchange
  uint32_t colS = 0, colQ = 0;                        // owner: exact column totals, kept across iterations
  uint32_t med_col = 0;                               // owner, kMedian: the column's lower median
  for (int64_t t = cluster_id_x(); t < P.total_tiles; t += nclusters) {
    const int b = (int)(t / P.tiles_per_beam);
    const int s0 = (int)(t % P.tiles_per_beam) * kStripCols;
    const int tw = min(kStripCols, P.S - s0);         // valid columns of this tile
    const uint8_t* gsrc = P.src + ((int64_t)b * C + c0) * P.stride + s0;   // row 0 of this CTA, column s0
    // ------------------------------------------------------------------ F1: load the CTA's rows
    if (kTensor) {
      // issued at the end of the previous tile (or before the loop)
    } else if (nload == 0) {
      if (tid == 0) mbar_arrive(&K->bar[0]);
    } else if (tid < nload) {
      uint32_t bytes = 0;
      for (int r = tid; r < nrows; r += kStripThreads) {
        const uint32_t off = (uint32_t)(reinterpret_cast<uintptr_t>(gsrc + (int64_t)r * P.stride) & 15);
        bytes += (off + (uint32_t)tw + 15u) & ~15u;
      }
      mbar_arrive_expect_tx(&K->bar[0], bytes);
      for (int r = tid; r < nrows; r += kStripThreads) {
        const uint8_t* g = gsrc + (int64_t)r * P.stride;
        const uint32_t off = (uint32_t)(reinterpret_cast<uintptr_t>(g) & 15);
        bulk_load(tile + (size_t)r * PW, g - off, (off + (uint32_t)tw + 15u) & ~15u, &K->bar[0]);
      }
    }
    mbar_wait(&K->bar[kWarpBox ? warp : kTensor ? cls : 0], phase);
    phase ^= 1;
    // While this tile is being processed, HBM delivers the NEXT tile into L2: the copies issued after this
    // tile's stores then come from L2 instead of waiting for DRAM behind those stores (6.6 -> 5.9 ms on config 4;
    // only with one CTA per SM: with two clusters per SM the prefetches get in each other's way, 7.0 -> 8.7 ms).
    if (kTensor && NW == 32 && tid < 4 && t + nclusters < P.total_tiles) {
      const int64_t tn = t + nclusters;
      const int bn = (int)(tn / P.tiles_per_beam);
      const int sn = (int)(tn % P.tiles_per_beam) * kStripCols;
      const int yn = (int)(((int64_t)bn * C + c0) >> 2);
      for (int y = 0; y < (Rq >> 2); y += P.box_rows) tma_prefetch_l2_2d(&maps.src[tid], sn, yn + y);
    }

    // rows warp + 16 i share the 16-byte phase of their global address: word offset of column s0 in them
    const int offw = (int)((reinterpret_cast<uintptr_t>(gsrc + (int64_t)warp * P.stride) & 15) >> 2);
    uint32_t* const col0 =
        kWarpBox ? tile + ((size_t)cls * (Rq >> 2) + (size_t)(warp >> 2) * ni) * PW + (P.off[cls] >> 2) + lane
        : kTensor ? tile + ((size_t)cls * (Rq >> 2) + (warp >> 2)) * PW + (P.off[cls] >> 2) + lane
                  : tile + (size_t)warp * PW + offw + lane;

    // one exchange: accumulators of all CTAs -> owners -> (lo, hi, r, packed constants) in every CTA
    auto exchange = [&](bool first, int itn) {
      sync_all();                                                   // A: accumulators complete everywhere
      if (owner) {
        // The owners' chain sits between two barriers with everybody else waiting: keep it short.  Without a
        // cluster everything is local shared memory; with one, all remote loads are issued before the first use.
        uint32_t s = 0, qq = 0;
        if (ncta == 1) {
          s = K->acc[buf][ocol];
          qq = K->acc[buf][kStripCols + ocol];
        } else {
          uint32_t vs[8], vq[8];
#pragma unroll
          for (uint32_t q = 0; q < 8; ++q) {
            vs[q] = 0; vq[q] = 0;
            if (q < ncta) {
              vs[q] = dsmem_ld_u32(dsmem_addr(&K->acc[buf][ocol], q));
              vq[q] = dsmem_ld_u32(dsmem_addr(&K->acc[buf][kStripCols + ocol], q));
            }
          }
#pragma unroll
          for (uint32_t q = 0; q < 8; ++q) { s += vs[q]; qq += vq[q]; }
        }
        if (first) { colS = s; colQ = qq; } else { colS += s; colQ += qq; }   // deltas are modulo 2^32
        int lo = 0, hi = 255;
        uint32_t r = 0;
        if (ocol < tw) {
          const uint64_t V = (uint64_t)C * colQ - (uint64_t)colS * colS;
          const U8Cut cut = make_cut_u8((uint32_t)C, colS, V, P.p[itn]);
          if (P.invC) {
            thread_bounds_u8_sqrt32(cut, P.invC, lo, hi, r);
          } else {
            thread_bounds_u8_sqrt(cut, lo, hi);
            r = rounded_mean_u8((uint32_t)C, colS);
          }
          if (kMedian && !first) r = med_col;                         // (first: the search below fills it in)
        }
        const int u = ocol & 3, slot = (u & 1) * 2 + (u >> 1);       // E.lo, O.lo, E.hi, O.hi
        const uint32_t neg = (0x10000u - ((uint32_t)lo << 8)) & 0xffffu;
        const uint32_t thr = lo > hi ? 0u : ((((uint32_t)(hi - lo)) << 8) | 0xffu);
        uint16_t* c16 = reinterpret_cast<uint16_t*>(&K->chk[ocol >> 2]);
        if (ncta == 1) {
          K->lo[ocol] = (uint8_t)lo;
          K->hi[ocol] = (uint8_t)hi;
          K->rr[ocol] = (uint8_t)r;
          c16[slot] = (uint16_t)neg;
          c16[4 + slot] = (uint16_t)thr;
        } else {
#pragma unroll
          for (uint32_t q = 0; q < 8; ++q) {
            if (q < ncta) {
              dsmem_st_u8(dsmem_addr(&K->lo[ocol], q), (uint32_t)lo);
              dsmem_st_u8(dsmem_addr(&K->hi[ocol], q), (uint32_t)hi);
              dsmem_st_u8(dsmem_addr(&K->rr[ocol], q), r);
              dsmem_st_u16(dsmem_addr(&c16[slot], q), neg);
              dsmem_st_u16(dsmem_addr(&c16[4 + slot], q), thr);
            }
          }
        }
      }
      sync_all();                                                   // B: bounds published everywhere
      if (tid < 2 * kStripCols) K->acc[buf][tid] = 0;               // nobody reads this buffer any more
      buf ^= 1;
    };

    uint8_t* const gds0 = P.dst + ((int64_t)b * C + c0 + row0) * P.stride + s0 + 4 * lane;
    const int64_t rstep = (int64_t)rowmul * P.stride;               // bytes between consecutive rows of this thread
    // Out of place, full-width tile: every word goes to the destination while the statistics read it (the stores
    // run under the other warps' copies and the exchange), and the rest of the tile's life is the in-place case:
    // only what an iteration repairs is written again (96 beams of config 4: 1.78 -> 1.27 ms; 12 beams: unchanged).
    const bool copy_early = kTensor && P.dst != P.src && tw == kStripCols;
    // ------------------------------------------------------------------ F2: column statistics
    if (ni > 0) {
      uint32_t S4[4] = {0, 0, 0, 0}, Q4[4] = {0, 0, 0, 0};
      const uint32_t* col = col0;
      uint8_t* ge = gds0;
      int i = 0;
#pragma unroll 2
      for (; i + 4 <= ni; i += 4, col += 4 * RS, ge += 4 * rstep) {
        const uint32_t a = col[0], bb = col[RS], c = col[2 * RS], d = col[3 * RS];
        if (copy_early) {
          *reinterpret_cast<uint32_t*>(ge) = a;
          *reinterpret_cast<uint32_t*>(ge + rstep) = bb;
          *reinterpret_cast<uint32_t*>(ge + 2 * rstep) = c;
          *reinterpret_cast<uint32_t*>(ge + 3 * rstep) = d;
        }
        const uint32_t ab_lo = prmt_b32(a, bb, 0x5140u), ab_hi = prmt_b32(a, bb, 0x7362u);
        const uint32_t cd_lo = prmt_b32(c, d, 0x5140u), cd_hi = prmt_b32(c, d, 0x7362u);
        const uint32_t t0 = prmt_b32(ab_lo, cd_lo, 0x5410u), t1 = prmt_b32(ab_lo, cd_lo, 0x7632u);
        const uint32_t t2 = prmt_b32(ab_hi, cd_hi, 0x5410u), t3 = prmt_b32(ab_hi, cd_hi, 0x7632u);
        S4[0] = __dp4a(t0, 0x01010101u, S4[0]); Q4[0] = __dp4a(t0, t0, Q4[0]);
        S4[1] = __dp4a(t1, 0x01010101u, S4[1]); Q4[1] = __dp4a(t1, t1, Q4[1]);
        S4[2] = __dp4a(t2, 0x01010101u, S4[2]); Q4[2] = __dp4a(t2, t2, Q4[2]);
        S4[3] = __dp4a(t3, 0x01010101u, S4[3]); Q4[3] = __dp4a(t3, t3, Q4[3]);
      }
      for (; i < ni; ++i, col += RS, ge += rstep) {
        const uint32_t w = col[0];
        if (copy_early) *reinterpret_cast<uint32_t*>(ge) = w;
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          const uint32_t x = (w >> (8 * u)) & 0xffu;
          S4[u] += x; Q4[u] += x * x;
        }
      }
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        smem_red_add(&K->acc[buf][4 * lane + u], S4[u]);
        smem_red_add(&K->acc[buf][kStripCols + 4 * lane + u], Q4[u]);
      }
    }
    if (P.n_thr > 0) exchange(true, 0);
    if (kMedian && P.n_thr > 0) {
      // T2m on the resident tile, once per column (the lower median does not change when samples are replaced by
      // it: DESIGN.md R22).  |median - mean| <= sigma always, so the search starts from [mean - sigma - 1, mean +
      // sigma + 1]; a step counts, per column, the samples above the probe value (packed compare, one byte counter
      // per column and thread) and halves the interval: the smallest v with #{x <= v} > rank is the lower median.
      const uint32_t rank_m = (uint32_t)(C - 1) >> 1;
      int vlo = 0, vhi = 0;
      if (owner && ocol < tw) {
        const uint64_t V = (uint64_t)C * colQ - (uint64_t)colS * colS;
        const float rc = 1.0f / (float)C;
        const float mu = (float)colS * rc, sg = sqrtf((float)V) * rc;
        vlo = max(0, (int)floorf(mu - sg) - 1);
        vhi = min(255, (int)ceilf(mu + sg) + 1);
      }
      while (true) {
        const bool active = owner && vlo < vhi;
        if (owner) { K->mid[ocol] = (uint8_t)((vlo + vhi) >> 1); K->cnt[ocol] = 0; }
        if (!__syncthreads_or(active)) break;                        // (also publishes the probes)
        if (ni > 0) {
          const uint32_t mid4 = reinterpret_cast<const uint32_t*>(K->mid)[lane];
          const uint32_t chiE = 0x7fff7fffu - prmt_b32(mid4, 0u, 0x4240u), chiO = 0x7fff7fffu - prmt_b32(mid4, 0u, 0x4341u);
          uint32_t above4 = 0;                                        // per column: samples > probe (ni <= 255)
          const uint32_t* col = col0;
#pragma unroll 4
          for (int i = 0; i < ni; ++i, col += RS)
            above4 += bytes_outside_cols(col[0], chiE, 0x80008000u, chiO, 0x80008000u) & 0x01010101u;
#pragma unroll
          for (int u = 0; u < 4; ++u) smem_red_add(&K->cnt[4 * lane + u], (above4 >> (8 * u)) & 0xffu);
        }
        __syncthreads();
        if (active) {
          const uint32_t le = (uint32_t)C - K->cnt[ocol];
          const int mid = (vlo + vhi) >> 1;
          if (le > rank_m) vhi = mid; else vlo = mid + 1;
        }
      }
      if (owner) { med_col = (uint32_t)vlo; K->rr[ocol] = (uint8_t)vlo; }
      __syncthreads();
    }

    // Tensor path, full-width tile: the LAST sweep writes the rows it finds clean straight from its registers
    // (F6 fused into F4: no second pass over shared memory for them); repaired rows are written by the repair.
    bool fused_store = false;
    const bool inplace = P.dst == P.src || copy_early;               // the destination already holds the input
    uint32_t dirty0 = 0u, dirty1 = 0u;                               // four-row steps some iteration has repaired
    // ------------------------------------------------------------------ F3..F5: thresholds, on chip
    for (int it = 0; it < P.n_thr; ++it) {
      const uint4 ck = K->chk[lane];
      const uint32_t lo4 = reinterpret_cast<const uint32_t*>(K->lo)[lane];
      const uint32_t hi4 = reinterpret_cast<const uint32_t*>(K->hi)[lane];
      const uint32_t r4 = reinterpret_cast<const uint32_t*>(K->rr)[lane];
      const uint32_t negE = ck.x, negO = ck.y, thrE = ck.z, thrO = ck.w;
      const uint32_t chiE = 0x7fff7fffu - prmt_b32(hi4, 0u, 0x4240u), cloE = 0x80008000u - prmt_b32(lo4, 0u, 0x4240u);
      const uint32_t chiO = 0x7fff7fffu - prmt_b32(hi4, 0u, 0x4341u), cloO = 0x80008000u - prmt_b32(lo4, 0u, 0x4341u);
      // a column with an empty kept interval (lo > hi) cuts every value: no packed test can say that,
      // so such a thread takes the exact path for all its words
      const bool slow = __vcmpgtu4(lo4, hi4) != 0u;
      const bool need_stats = it + 1 < P.n_thr;

      uint32_t cnt4 = 0, sxE = 0, sxO = 0, sq[4] = {0, 0, 0, 0};   // per-column deltas of this thread, packed
      auto fix_word = [&](uint32_t* ptr, uint32_t w, int i) {
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
          uint8_t* fl = P.flags + ((int64_t)b * C + c0 + row0 + rowmul * i) * P.S + s0 + 4 * lane;
#pragma unroll
          for (int u = 0; u < 4; ++u)
            if ((m >> (8 * u)) & 1u) fl[u] = 1;
        }
      };
      auto hit = [&](uint32_t w) {
        return slow || __viaddmax_u16x2(w, negO, thrO) != thrO || __viaddmax_u16x2(w << 8, negE, thrE) != thrE;
      };
      // F4: sweep first (one bit per four-row step that holds an outlier), repair afterwards over the set bits:
      // a warp step covers 512 bytes, so at k = 3 nearly every step has SOME lane with an outlier, and a repair
      // inside the sweep would make every lane pay for it at every step.
      {
        uint32_t* col = col0;
        auto step_hits = [&](const uint32_t* c) {        // packed test of four rows of this thread's word column
          const uint32_t w0 = c[0], w1 = c[RS], w2 = c[2 * RS], w3 = c[3 * RS];
          uint32_t aO = __viaddmax_u16x2(w0, negO, 0u), aE = __viaddmax_u16x2(w0 << 8, negE, 0u);
          uint32_t bO = __viaddmax_u16x2(w1, negO, 0u), bE = __viaddmax_u16x2(w1 << 8, negE, 0u);
          aO = __viaddmax_u16x2(w2, negO, aO); aE = __viaddmax_u16x2(w2 << 8, negE, aE);
          bO = __viaddmax_u16x2(w3, negO, bO); bE = __viaddmax_u16x2(w3 << 8, negE, bE);
          aO = __vimax3_u16x2(aO, bO, thrO); aE = __vimax3_u16x2(aE, bE, thrE);
          return ((aO ^ thrO) | (aE ^ thrE)) != 0u;
        };
        // one bit per step in two 32-bit words (a running bit instead of a 64-bit variable shift per step)
        const int n4 = ni >> 2, nA = min(n4, 32);
        uint32_t hm0 = 0u, hm1 = 0u, bit = 1u;
        int st4 = 0;
        const bool fuse = kTensor && !need_stats && tw == kStripCols;
        if (fuse) {
          fused_store = true;
          // In place a clean step that no earlier iteration repaired still holds the input: nothing to write.
          auto step_store = [&](const uint32_t* c, uint8_t* g, bool skip) {   // the same test; clean rows go out at once
            const uint32_t w0 = c[0], w1 = c[RS], w2 = c[2 * RS], w3 = c[3 * RS];
            uint32_t aO = __viaddmax_u16x2(w0, negO, 0u), aE = __viaddmax_u16x2(w0 << 8, negE, 0u);
            uint32_t bO = __viaddmax_u16x2(w1, negO, 0u), bE = __viaddmax_u16x2(w1 << 8, negE, 0u);
            aO = __viaddmax_u16x2(w2, negO, aO); aE = __viaddmax_u16x2(w2 << 8, negE, aE);
            bO = __viaddmax_u16x2(w3, negO, bO); bE = __viaddmax_u16x2(w3 << 8, negE, bE);
            aO = __vimax3_u16x2(aO, bO, thrO); aE = __vimax3_u16x2(aE, bE, thrE);
            const bool h = ((aO ^ thrO) | (aE ^ thrE)) != 0u;
            if (!h && !skip) {
              *reinterpret_cast<uint32_t*>(g) = w0;
              *reinterpret_cast<uint32_t*>(g + rstep) = w1;
              *reinterpret_cast<uint32_t*>(g + 2 * rstep) = w2;
              *reinterpret_cast<uint32_t*>(g + 3 * rstep) = w3;
            }
            return h;
          };
          uint8_t* g = gds0;
#pragma unroll 2
          for (; st4 < nA; ++st4, col += 4 * RS, g += 4 * rstep, bit <<= 1)
            if (step_store(col, g, inplace && (dirty0 & bit) == 0u)) hm0 |= bit;
          bit = 1u;
          for (; st4 < n4; ++st4, col += 4 * RS, g += 4 * rstep, bit <<= 1)
            if (step_store(col, g, inplace && (dirty1 & bit) == 0u)) hm1 |= bit;
        } else {
#pragma unroll 4
          for (; st4 < nA; ++st4, col += 4 * RS, bit <<= 1)
            if (step_hits(col)) hm0 |= bit;
          bit = 1u;
          for (; st4 < n4; ++st4, col += 4 * RS, bit <<= 1)
            if (step_hits(col)) hm1 |= bit;
        }
        unsigned long long hm = ((unsigned long long)hm1 << 32) | hm0;
        dirty0 |= slow ? ~0u : hm0;                                   // steps this iteration may modify
        dirty1 |= slow ? ~0u : hm1;
        int i = 4 * n4;
        for (; i < ni; ++i, col += RS) {
          fix_word(col, col[0], i);
          if (fuse) *reinterpret_cast<uint32_t*>(gds0 + (int64_t)i * rstep) = col[0];
        }
        const int nsteps = ni >> 2;
        if (slow) hm = nsteps < 64 ? (1ull << nsteps) - 1ull : ~0ull;
        while (hm) {
          const int st = __ffsll((long long)hm) - 1;
          hm &= hm - 1ull;
          uint32_t* c4 = col0 + (size_t)st * 4 * RS;
          const uint32_t w0 = c4[0], w1 = c4[RS], w2 = c4[2 * RS], w3 = c4[3 * RS];
          if (hit(w0)) fix_word(c4, w0, 4 * st);
          if (hit(w1)) fix_word(c4 + RS, w1, 4 * st + 1);
          if (hit(w2)) fix_word(c4 + 2 * RS, w2, 4 * st + 2);
          if (hit(w3)) fix_word(c4 + 3 * RS, w3, 4 * st + 3);
          if (fuse) {
            uint8_t* g = gds0 + (int64_t)st * 4 * rstep;
            *reinterpret_cast<uint32_t*>(g) = c4[0];
            *reinterpret_cast<uint32_t*>(g + rstep) = c4[RS];
            *reinterpret_cast<uint32_t*>(g + 2 * rstep) = c4[2 * RS];
            *reinterpret_cast<uint32_t*>(g + 3 * rstep) = c4[3 * RS];
          }
        }
      }
      if ((need_stats || P.counts) && __any_sync(FULL, cnt4 != 0u)) {
        uint32_t cnt = 0;
        if (cnt4) {
#pragma unroll
          for (int u = 0; u < 4; ++u) {
            const uint32_t c = (cnt4 >> (8 * u)) & 0xffu, r = (r4 >> (8 * u)) & 0xffu;
            const uint32_t sx = ((u & 1) ? sxO : sxE) >> (16 * (u >> 1)) & 0xffffu;
            cnt += c;
            if (need_stats && c) {                       // modulo 2^32: the column totals stay below 2^32
              smem_red_add(&K->acc[buf][4 * lane + u], c * r - sx);
              smem_red_add(&K->acc[buf][kStripCols + 4 * lane + u], c * r * r - sq[u]);
            }
          }
        }
        if (P.counts) {
          cnt = __reduce_add_sync(FULL, cnt);
          if (lane == 0 && cnt) atomicAdd(&P.counts[it], (unsigned long long)cnt);
        }
      }
      if (need_stats) exchange(false, it + 1);
    }

    // ------------------------------------------------------------------ F6: store the CTA's rows
    if (kTensor) {
      // a warp writes the 128-byte segment of one row per step: 32 lanes x one 32-bit word.  Only this warp
      // ever touched its rows, so no barrier is needed before the store.
      uint8_t* gd = gds0;
      const uint32_t* col = col0;
      const int nb = fused_store ? 0 : tw - 4 * lane;   // valid bytes of this lane's word (0: already written)
      if (nb >= 4) {
#pragma unroll 4
        for (int i = 0; i < ni; ++i, col += RS, gd += rstep)
          *reinterpret_cast<uint32_t*>(gd) = col[0];
      } else if (nb > 0) {
        for (int i = 0; i < ni; ++i, col += RS, gd += rstep) {
          const uint32_t w = col[0];
          for (int u = 0; u < nb; ++u) gd[u] = (uint8_t)(w >> (8 * u));
        }
      }
      // the class's rows are free once its NW / 4 warps are here: fetch the class's rows of the next tile
      fence_proxy_async_smem();
      if (kWarpBox) {                               // the warp's rows are free: fetch its rows of the next tile
        __syncwarp();
        if (lane == 0 && t + nclusters < P.total_tiles) issue_warp_load(t + nclusters);
      } else {
        asm volatile("bar.sync %0, %1;" ::"r"(1 + cls), "n"(32 * (NW / 4)) : "memory");
        if (warp == cls && lane == 0 && t + nclusters < P.total_tiles) issue_class_load(t + nclusters, cls);
      }
    } else {
      fence_proxy_async_smem();                     // generic-proxy writes of the repair -> async proxy
      __syncthreads();
      uint8_t* gdst = P.dst + ((int64_t)b * C + c0) * P.stride + s0;
      bool issued = false;
      for (int r = tid; r < nrows; r += kStripThreads) {
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
      __syncthreads();
    }
  }
  bulk_wait_all<0>();
  if (ncta > 1) cluster_sync_all();                 // no CTA leaves while a peer may still access its shared memory
}

}  // namespace rfim
