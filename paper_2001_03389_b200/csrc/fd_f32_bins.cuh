// fd_f32_bins.cuh -- frequency-domain sigma cut (FDSC, Fig. 3) for float32 dynamic spectra WITH
// the paper's per-bin mean correction (PAPER.md:102 step 1, :126), mean or lower-median replacement:
// the resident-tile kernel of fd_f32_tile.cuh with bins.
//
// A tile is ALL channels x COLS consecutive samples of one beam, brought into shared memory by 2-D TMA tensor copies
// exactly as in fd_f32_tile.cuh (same tensor maps, boxes, parameter block).  What differs is who owns what: there a
// thread reads rows w, w + NVW, ... of its column (coalesced across the lanes of a row, the warps meet in shared
// memory for every sum); here a thread owns WHOLE BINS of its column -- bins v, v + NVW, ... for virtual warp v -- so
// that everything the definition asks per bin stays in registers:
//   step 1  bin mean m_b and sum (x - m_b)^2 in ONE fp64 pass around a pivot (the bin's first channel), redone the
//           long way when the pivot is the outlier; odd virtual warps visit the rows of a bin pairwise swapped so that
//           the two half-warps of a hardware warp never hit the same banks;
//   step 2  A = sum (x - m_b), B = sum (x - m_b)^2 over the thread's bins; one shared-memory reduction per column
//           gives mu' = A / C and sigma'^2 = B / C - mu'^2 (the corrected values are centred: nothing cancels);
//   step 3  flag <=> |x - (m_b + mu')| > k sigma' in fp64, decided by two float bounds per bin that are equivalent to
//           that test (f32_bounds), so the scan is two float compares per sample; a flagged sample's ORIGINAL
//           value is replaced by (float) m_b or by the bin's lower median, both taken from the snapshot at the start of
//           the iteration (the bin is scanned for flags first, replaced afterwards; the median -- rank floor((nb-1)/2)
//           by counting, O(nb^2) on a bin that has a flagged sample, one bin in six at 2.75 sigma -- before the first
//           replacement).
// Every iteration recomputes steps 1-3 from the resident tile (two passes over shared memory, no deltas).
// In place only replaced samples are written; out of place the tile leaves by TMA tensor stores.
#pragma once

#include <cuda.h>

#include "common.cuh"
#include "td_f32.cuh"        // f32_bounds
#include "fd_f32_tile.cuh"   // FdF32TileMaps / FdF32TileParams, FtCtrl, ft_tma_* helpers

namespace rfim {

constexpr int kFbKeep = 3;                           // bin means a thread keeps in registers between steps 2 and 3

template <int COLS>
__global__ void __launch_bounds__(kFtThreads, COLS == 32 ? 1 : 2) fd_f32_bins_kernel(const __grid_constant__ FdF32TileMaps maps,
                                                                                     const FdF32TileParams P, const int nb) {
  extern __shared__ __align__(128) uint8_t smem[];
  constexpr int NVW = FtCtrl<COLS>::NVW;                                // virtual warps of COLS lanes
  float* const tile = reinterpret_cast<float*>(smem);                   // [C][COLS]
  FtCtrl<COLS>* const K = reinterpret_cast<FtCtrl<COLS>*>(smem + (size_t)P.C * COLS * 4);
  const int tid = threadIdx.x;
  const int lane = tid & (COLS - 1);                                    // column of the tile
  const int vw = tid / COLS;                                            // virtual warp: bins vw, vw + NVW, ...
  const int hwlane = tid & 31;
  const int C = P.C, nbins = C / nb;
  const double rn = 1.0 / (double)C, rnb = (double)nb;
  // 16-column tiles: the two half-warps of a hardware warp work on different bins whose rows, nb apart, fall into the
  // same banks when nb is even; the odd half therefore visits the rows of a bin pairwise swapped (1, 0, 3, 2, ...):
  // step j is row j ^ 1, reached through two base pointers one row up / down, so that no step costs an instruction
  const int sw = ((COLS < 32) && (vw & 1) && (nb & 1) == 0) ? 1 : 0;
  const int skew = sw * COLS;
  if (tid == 0) {
    for (int i = 0; i < P.nboxes; ++i) mbar_init(&K->bar[i], 1);
    fence_mbar_init();
    asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(&maps.src)) : "memory");
    if (P.copy) asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(&maps.dst)) : "memory");
  }
  __syncthreads();

  // sum of two doubles per column over the virtual warps (result in every thread of the column)
  // (16 columns: the two virtual warps of a hardware warp hold the same columns and meet by a shuffle first)
  constexpr int NRED = COLS == 16 ? NVW / 2 : NVW;
  auto col_sum2 = [&](double& a, double& b) {
    if (COLS == 16) {
      a += __shfl_xor_sync(FULL, a, 16);
      b += __shfl_xor_sync(FULL, b, 16);
      if ((vw & 1) == 0) { K->red[vw >> 1][lane][0] = a; K->red[vw >> 1][lane][1] = b; }
    } else {
      K->red[vw][lane][0] = a;
      K->red[vw][lane][1] = b;
    }
    __syncthreads();
    a = 0.0; b = 0.0;
#pragma unroll
    for (int w = 0; w < NRED; ++w) { a += K->red[w][lane][0]; b += K->red[w][lane][1]; }
    __syncthreads();
  };
  auto col_sum_u32 = [&](uint32_t v) {
    if (COLS == 16) {
      v += __shfl_xor_sync(FULL, v, 16);
      if ((vw & 1) == 0) K->cred[vw >> 1][lane] = v;
    } else {
      K->cred[vw][lane] = v;
    }
    __syncthreads();
    uint32_t s = 0;
#pragma unroll
    for (int w = 0; w < NRED; ++w) s += K->cred[w][lane];
    __syncthreads();
    return s;
  };
  // row of step j (0 .. nb - 1) of a bin that starts at row r0
  auto row_of = [&](int r0, int j) { return r0 + (j ^ sw); };

  uint32_t phase = 0;
  for (int64_t t = blockIdx.x; t < P.total_tiles; t += gridDim.x) {
    const int b = (int)(t / P.tiles_per_beam);
    const int s0 = (int)(t % P.tiles_per_beam) * COLS;
    const int tw = min(COLS, P.S - s0);
    const bool valid = lane < tw;
    const int y0 = b * C;
    // ------------------------------------------------------------------ F1: load (every box, then everybody waits)
    if (tid == 0) {
      for (int i = 0; i < P.nboxes; ++i) {
        mbar_arrive_expect_tx(&K->bar[i], (uint32_t)P.box_rows * COLS * 4u);
        ft_tma_load_2d(tile + (size_t)i * P.box_rows * COLS, &maps.src, s0, y0 + i * P.box_rows, &K->bar[i]);
      }
    }
    for (int i = 0; i < P.nboxes; ++i) mbar_wait(&K->bar[i], phase);

    float* const gcol = P.dst + (int64_t)y0 * P.stride + s0 + lane;
    for (int it = 0; it < P.n_thr; ++it) {
      // ---------------------------------------------------------------- steps 1 + 2: bin means, corrected sums
      // One pass per bin around a pivot (the bin's first channel): Sd = sum (x - x0), Sdd = sum (x - x0)^2 in fp64,
      // m_b = x0 + Sd / nb, sum (x - m_b)^2 = Sdd - Sd^2 / nb.  Exact enough unless the pivot sits far outside the
      // bin's spread (it is the outlier): then the bin is summed the long way, mean first.
      double A = 0.0, B = 0.0;
      double mkeep[kFbKeep];                                           // means of the thread's first bins, for step 3
#pragma unroll
      for (int i = 0; i < kFbKeep; ++i) mkeep[i] = 0.0;
      auto bin_stats = [&](int r0, double& m, double& a, double& q) {
        const double x0 = (double)tile[r0 * COLS + lane];
        const float* const pe = tile + r0 * COLS + lane + skew;       // even steps
        const float* const po = pe - 2 * skew;                        // odd steps
        double sd = 0.0, sdd = 0.0;
        int j = 0;
#pragma unroll 4
        for (; j + 2 <= nb; j += 2) {
          const double d0 = (double)pe[j * COLS] - x0, d1 = (double)po[(j + 1) * COLS] - x0;
          sd += d0; sdd = fma(d0, d0, sdd);
          sd += d1; sdd = fma(d1, d1, sdd);
        }
        if (j < nb) {                                                  // (odd nb: no swap)
          const double d = (double)pe[j * COLS] - x0;
          sd += d; sdd = fma(d, d, sdd);
        }
        const double md = sd / rnb;
        m = x0 + md;
        a = fma(-rnb, md, sd);                                         // sum (x - m_b): rounding residue
        q = fma(-sd, md, sdd);
        if (!(q > 1e-6 * sdd)) {                                       // cancellation (or a constant bin): the long way
          double s1 = 0.0;
          for (int j = 0; j < nb; ++j) s1 += (double)tile[row_of(r0, j) * COLS + lane];
          m = s1 / rnb;
          a = 0.0; q = 0.0;
          for (int j = 0; j < nb; ++j) {
            const double d = (double)tile[row_of(r0, j) * COLS + lane] - m;
            a += d; q = fma(d, d, q);
          }
        }
      };
      if (valid) {
        int own = 0;
        for (int bn = vw; bn < nbins; bn += NVW, ++own) {
          double m, a, q;
          bin_stats(bn * nb, m, a, q);
#pragma unroll
          for (int i = 0; i < kFbKeep; ++i)
            if (own == i) mkeep[i] = m;
          A += a; B += q;
        }
      }
      col_sum2(A, B);
      const double mu = A * rn;
      double var = B * rn - mu * mu;
      if (!(var > 0.0)) var = 0.0;
      const double cut = P.k[it] * sqrt(var);
      // ---------------------------------------------------------------- step 3: flag, replace (own bins only)
      // flag <=> |x - (m_b + mu')| > k sigma' in fp64, taken as two float bounds per bin that decide exactly that
      // (f32_bounds): the scan of a bin is two float compares per sample
      uint32_t cnt = 0;
      if (valid) {
        int own = 0;
        for (int bn = vw; bn < nbins; bn += NVW, ++own) {
          const int r0 = bn * nb;
          double m = 0.0;
          if (own < kFbKeep) {
#pragma unroll
            for (int i = 0; i < kFbKeep; ++i)
              if (own == i) m = mkeep[i];
          } else {                                                     // (many small bins: summed again)
            double a, q;
            bin_stats(r0, m, a, q);
          }
          float t_lo, t_hi;
          f32_bounds(m + mu, cut, t_lo, t_hi);
          // scan the snapshot first: bit j <=> the sample of step j is flagged (nb <= 64: host-checked)
          {
            const float* const pe = tile + r0 * COLS + lane + skew;
            const float* const po = pe - 2 * skew;
            uint32_t f0 = 0u, f1 = 0u;                                  // steps 0..31 and 32..63
            int j = 0;
#pragma unroll 4
            for (; j + 2 <= nb; j += 2) {
              const float v0 = pe[j * COLS], v1 = po[(j + 1) * COLS];
              const uint32_t h = ((v0 > t_hi || v0 < t_lo) ? 1u : 0u) | ((v1 > t_hi || v1 < t_lo) ? 2u : 0u);
              if (j < 32) f0 |= h << (j & 31); else f1 |= h << (j & 31);
            }
            if (j < nb) {
              const float v = pe[j * COLS];
              const uint32_t h = (v > t_hi || v < t_lo) ? 1u : 0u;
              if (j < 32) f0 |= h << (j & 31); else f1 |= h << (j & 31);
            }
            unsigned long long fm = ((unsigned long long)f1 << 32) | f0;
            if (fm == 0ull) continue;
            float rv = (float)m;
            if (P.policy != 0) {
              // lower median of the bin's snapshot: the element with exactly floor((nb - 1) / 2) elements that are
              // smaller, or equal and earlier
              const uint32_t want = (uint32_t)(nb - 1) >> 1;
              for (int i = 0; i < nb; ++i) {
                const float e = tile[(r0 + i) * COLS + lane];
                uint32_t rank = 0;
                for (int k2 = 0; k2 < nb; ++k2) {
                  const float o = tile[(r0 + k2) * COLS + lane];
                  rank += (o < e) || (o == e && k2 < i);
                }
                if (rank == want) { rv = e; break; }
              }
            }
            while (fm) {
              const int j = __ffsll((long long)fm) - 1;
              fm &= fm - 1ull;
              const int r = row_of(r0, j);
              tile[r * COLS + lane] = rv;
              if (!P.copy) gcol[(int64_t)r * P.stride] = rv;
              if (P.flags) P.flags[((int64_t)y0 + r) * P.S + s0 + lane] = 1;
              ++cnt;
            }
          }
        }
      }
      if (P.counts) {
        const uint32_t total = col_sum_u32(cnt);
        if (tid < 32) {                                                 // (one copy of every column's total)
          const uint32_t all = __reduce_add_sync(FULL, hwlane < COLS ? total : 0u);
          if (hwlane == 0 && all) atomicAdd(&P.counts[it], (unsigned long long)all);
        }
      }
      // (no barrier needed between iterations beyond col_sum2's: a thread touches only its own bins)
    }

    // ------------------------------------------------------------------ F6: store (out of place), next tile
    fence_proxy_async_smem();                          // generic-proxy accesses of the tile before the async proxy's
    if (P.copy) {
      __syncthreads();
      if (tid == 0) {
        for (int i = 0; i < P.nboxes; ++i)
          ft_tma_store_2d(&maps.dst, s0, y0 + i * P.box_rows, tile + (size_t)i * P.box_rows * COLS);
        bulk_commit();
        bulk_wait_read<0>();
      }
    }
    __syncthreads();
    phase ^= 1;
  }
  if (P.copy && tid == 0) bulk_wait_all<0>();
}

}  // namespace rfim
