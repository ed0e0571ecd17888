// fd_f32_tile.cuh -- frequency-domain sigma cut (FDSC, Fig. 3) for float32 dynamic spectra, one
// bin, mean or lower-median replacement: the resident-tile kernel.
//
// A tile is ALL channels x 32 consecutive samples of one beam (1536 x 128 bytes = 192 KB), brought into shared memory
// by a handful of 2-D TMA tensor copies (boxes of 32 floats x up to 256 rows, one mbarrier each, so the statistics
// start on the first box while the others are still in flight).  One CTA of 16 warps per SM; lane = column, warp w
// owns rows w, w + 16, ...: a warp reads 32 consecutive floats of a row (no bank conflicts).
//   F2  fp64 sums per column around a pivot (the column's first channel), A = sum (x - c), B = sum (x - c)^2, the 16
//       warps meet in shared memory; re-taken around the mean when B/n - (A/n)^2 would cancel (td_f32.cuh).
//   F3  mu, sigma, cut = k sigma in fp64 -> two float bounds equal to the fp64 test (f32_bounds), per column, by
//       every warp for its lanes (cheaper than publishing them).
//   F4  one sweep over the resident tile: flagged samples are replaced in shared memory (and, in place, in global
//       memory: nothing else is written), fp64 deltas give the statistics of the next iteration (F5).
//   T2m lower median of a column by bracketing (two pivots per counting pass, then gather <= 32 candidates and
//       rank), once per column: replacing samples by the lower median never changes it (td_f32_fast.cuh).
//   F6  out of place the whole tile is written back by TMA tensor stores.
// With one bin the paper's mean-corrected statistics are the column's own mean and population sigma (the bin mean
// is the column mean, the corrected values have mean zero up to rounding).
#pragma once

#include <cuda.h>

#include "common.cuh"
#include "td_f32.cuh"        // f32_bounds, f32_key, f32_next_up / down
#include "td_f32_fast.cuh"   // f32f_le_mask

namespace rfim {

constexpr int kFtWarps = 16;
constexpr int kFtThreads = 32 * kFtWarps;
constexpr int kFtCap = 32;
constexpr int kFtMaxBoxes = 8;

struct FdF32TileMaps { CUtensorMap src, dst; };

struct FdF32TileParams {
  const float* src;
  float* dst;
  int64_t stride;
  int beams, C, S;
  int n_thr, policy;
  double k[16];
  uint8_t* flags;
  unsigned long long* counts;
  int box_rows, nboxes;            // C = box_rows * nboxes
  int tiles_per_beam;
  int64_t total_tiles;
  int copy;                        // out of place
};

// COLS = samples per tile: 32 (one CTA per SM) or 16 (tiles of half the size, two CTAs per SM whose loads, sweeps
// and stores overlap).  A row of the tile is read by COLS lanes: a warp covers 32 / COLS rows at a time and counts as
// 32 / COLS "virtual warps" of COLS lanes; 512 threads = kFtWarps * 32 / COLS virtual warps.
template <int COLS>
struct __align__(16) FtCtrl {
  static constexpr int NVW = kFtWarps * 32 / COLS;
  double red[NVW][COLS][2];
  uint32_t cred[NVW][COLS];
  uint16_t list[kFtCap][COLS];
  int ln[COLS];
  float med[COLS];
  uint64_t bar[kFtMaxBoxes];
};
template <int COLS>
__host__ __device__ inline size_t fd_f32_tile_smem_bytes(int C) {
  return (size_t)C * COLS * 4 + sizeof(FtCtrl<COLS>);
}

__device__ __forceinline__ void ft_tma_load_2d(void* smem_dst, const CUtensorMap* map, int x, int y, uint64_t* bar) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
      ::"r"(smem_addr(smem_dst)), "l"(reinterpret_cast<uint64_t>(map)), "r"(x), "r"(y), "r"(smem_addr(bar))
      : "memory");
}
__device__ __forceinline__ void ft_tma_store_2d(const CUtensorMap* map, int x, int y, const void* smem_src) {
  asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.tile.bulk_group [%0, {%1, %2}], [%3];" ::"l"(
                   reinterpret_cast<uint64_t>(map)),
               "r"(x), "r"(y), "r"(smem_addr(smem_src))
               : "memory");
}

template <int COLS>
__global__ void __launch_bounds__(kFtThreads, COLS == 32 ? 1 : 2) fd_f32_tile_kernel(const __grid_constant__ FdF32TileMaps maps,
                                                                                     const FdF32TileParams P) {
  extern __shared__ __align__(128) uint8_t smem[];
  constexpr int kFtCols = COLS;
  constexpr int NVW = FtCtrl<COLS>::NVW;                                // virtual warps (rows read side by side)
  float* const tile = reinterpret_cast<float*>(smem);                   // [C][COLS]
  FtCtrl<COLS>* const K = reinterpret_cast<FtCtrl<COLS>*>(smem + (size_t)P.C * kFtCols * 4);
  const int tid = threadIdx.x;
  const int lane = tid & (COLS - 1);                                    // column of the tile
  const int warp = tid / COLS;                                          // virtual warp: rows warp, warp + NVW, ...
  const int hwlane = tid & 31;
  const int C = P.C;
  const double rn = 1.0 / (double)C;
  const float inf = __int_as_float(0x7f800000);
  if (tid == 0) {
    for (int i = 0; i < P.nboxes; ++i) mbar_init(&K->bar[i], 1);
    fence_mbar_init();
    asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(&maps.src)) : "memory");
    if (P.copy) asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(&maps.dst)) : "memory");
  }
  __syncthreads();

  // sum of two doubles per column over the 16 warps (result in every thread of the column)
  // (16 columns: the two virtual warps of a hardware warp hold the same columns and meet by a shuffle first, which
  // halves the partial sums every thread has to add up)
  constexpr int NRED = COLS == 16 ? NVW / 2 : NVW;
  auto col_sum2 = [&](double& a, double& b) {
    if (COLS == 16) {
      a += __shfl_xor_sync(FULL, a, 16);
      b += __shfl_xor_sync(FULL, b, 16);
      if ((warp & 1) == 0) { K->red[warp >> 1][lane][0] = a; K->red[warp >> 1][lane][1] = b; }
    } else {
      K->red[warp][lane][0] = a;
      K->red[warp][lane][1] = b;
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
      if ((warp & 1) == 0) K->cred[warp >> 1][lane] = v;
    } else {
      K->cred[warp][lane] = v;
    }
    __syncthreads();
    uint32_t s = 0;
#pragma unroll
    for (int w = 0; w < NRED; ++w) s += K->cred[w][lane];
    __syncthreads();
    return s;
  };

  uint32_t phase = 0;
  for (int64_t t = blockIdx.x; t < P.total_tiles; t += gridDim.x) {
    const int b = (int)(t / P.tiles_per_beam);
    const int s0 = (int)(t % P.tiles_per_beam) * kFtCols;
    const int tw = min(kFtCols, P.S - s0);
    const bool valid = lane < tw;
    const int y0 = b * C;
    // ------------------------------------------------------------------ F1: load
    if (tid == 0) {
      for (int i = 0; i < P.nboxes; ++i) {
        mbar_arrive_expect_tx(&K->bar[i], (uint32_t)P.box_rows * kFtCols * 4u);
        ft_tma_load_2d(tile + (size_t)i * P.box_rows * kFtCols, &maps.src, s0, y0 + i * P.box_rows, &K->bar[i]);
      }
    }
    // ------------------------------------------------------------------ F2: statistics
    mbar_wait(&K->bar[0], phase);
    double piv = (double)tile[lane];                                     // row 0 of the column
    double A = 0.0, B = 0.0;
    // rows warp, warp + NVW, ... of the column, eight per trip at compile-time offsets; the first pass follows the
    // tensor boxes as they land (one wait per box instead of a check per row)
    constexpr int RSTEP = NVW * kFtCols;                               // floats between consecutive rows of a thread
    const float* const pcol = tile + warp * kFtCols + lane;
    const int nrows = C > warp ? (C - warp + NVW - 1) / NVW : 0;       // rows of this thread
    auto sums = [&](bool first) {
      double A0 = 0.0, B0 = 0.0, A1 = 0.0, B1 = 0.0;
      int i = 0;
      for (int box = 0; box < P.nboxes; ++box) {
        if (first && box > 0) mbar_wait(&K->bar[box], phase);
        // rows of this thread below the end of the box: warp + NVW i < (box + 1) box_rows
        const int lim = box + 1 == P.nboxes ? nrows : min(nrows, max(0, ((box + 1) * P.box_rows - warp + NVW - 1) / NVW));
        const float* q = pcol + (size_t)i * RSTEP;
#pragma unroll 1
        for (; i + 8 <= lim; i += 8, q += 8 * RSTEP) {
#pragma unroll
          for (int u = 0; u < 8; u += 2) {
            const double d0 = (double)q[u * RSTEP] - piv, d1 = (double)q[(u + 1) * RSTEP] - piv;
            A0 += d0; B0 = fma(d0, d0, B0);
            A1 += d1; B1 = fma(d1, d1, B1);
          }
        }
        for (; i < lim; ++i, q += RSTEP) {
          const double d0 = (double)q[0] - piv;
          A0 += d0; B0 = fma(d0, d0, B0);
        }
      }
      A = A0 + A1; B = B0 + B1;
      col_sum2(A, B);
    };
    auto cancels = [&]() {
      const double am = A * rn, m2 = B * rn;
      return m2 - am * am < 1e-6 * m2;
    };
    sums(true);
    if (__syncthreads_or(valid && cancels())) {
      if (cancels()) piv += A * rn;
      sums(false);
    }

    // ------------------------------------------------------------------ T2m: lower median of every column, once
    float median = 0.0f;
    if (P.policy != 0 && P.n_thr > 0) {
      const double am = A * rn;
      const float muf = (float)(piv + am);
      double var = B * rn - am * am;
      if (!(var > 0.0)) var = 0.0;
      const float sigf = (float)sqrt(var);
      const uint32_t rho = (uint32_t)(C - 1) >> 1;
      float a = -inf, bb = inf;
      uint32_t ca = 0, cb = (uint32_t)C;
      float R = 3.2f * sigf * rsqrtf((float)C);
      float p1 = muf - R, p2 = muf + R;
      bool done = !valid;
      float result = 0.0f;
      bool searching = valid && cb - ca > (uint32_t)kFtCap;
      for (int pass = 0; pass < 64 && __syncthreads_or(searching); ++pass) {
        if (!(p1 > a)) p1 = a;
        if (!(p2 < bb)) p2 = bb;
        if (!(p1 <= p2)) p1 = p2;
        uint32_t c1 = 0, c2 = 0;
        {
          const float* q = pcol;
          int i = 0;
#pragma unroll 1
          for (; i + 8 <= nrows; i += 8, q += 8 * RSTEP) {
#pragma unroll
            for (int u = 0; u < 8; ++u) {
              const float v = q[u * RSTEP];
              c1 -= f32f_le_mask(v, p1);
              c2 -= f32f_le_mask(v, p2);
            }
          }
          for (; i < nrows; ++i, q += RSTEP) {
            const float v = q[0];
            c1 -= f32f_le_mask(v, p1);
            c2 -= f32f_le_mask(v, p2);
          }
        }
        const uint32_t packed = col_sum_u32(c1 | (c2 << 16));            // C <= 2^15 (host-checked)
        if (searching) {
          c1 = packed & 0xffffu;
          c2 = packed >> 16;
          if (rho < c1) { bb = p1; cb = c1; }
          else if (rho < c2) { a = p1; ca = c1; bb = p2; cb = c2; }
          else { a = p2; ca = c2; }
          const uint32_t m = cb - ca;
          if (m <= (uint32_t)kFtCap) {
            searching = false;
          } else if (a > -inf && bb < inf) {
            const float w = bb - a;
            const float f = ((float)(rho - ca) + 0.5f) / (float)m;
            const float dev = (2.0f * sqrtf(f * (1.0f - f) * (float)m) + 1.0f) / (float)m;
            p1 = a + w * fmaxf(f - dev, 0.0f);
            p2 = a + w * fminf(f + dev, 1.0f);
            if (!(p1 > a)) p1 = f32_next_up(a);
            if (!(p2 < bb)) p2 = f32_next_down(bb);
            if (!(p2 >= p1)) p2 = p1;
            if (!(w <= 3.0e38f)) searching = false;                      // -> key bisection
            else if (!(p1 < bb)) { searching = false; done = true; result = bb; }   // neighbouring floats: all == b
          } else if (bb == inf && a == -inf) {
            R *= 2.0f;
            p1 = muf - R; p2 = muf + R;
          } else if (bb == inf) {
            R *= 4.0f;
            p1 = a + R; p2 = a + 4.0f * R;
            if (!(p1 > a)) { p1 = 3.402823466e38f; p2 = 3.402823466e38f; }
            if (!(p2 < inf)) p2 = 3.402823466e38f;
          } else {
            R *= 4.0f;
            p2 = bb - R; p1 = bb - 4.0f * R;
            if (!(p2 < bb)) { p1 = -3.402823466e38f; p2 = -3.402823466e38f; }
            if (!(p1 > -inf)) p1 = -3.402823466e38f;
          }
        }
      }
      const bool bisect = valid && !done && cb - ca > (uint32_t)kFtCap;
      if (__syncthreads_or(bisect)) {                                    // last resort: 32 halvings of the key range
        uint32_t klo = 0u, khi = 0xffffffffu;
        for (int step = 0; step < 32; ++step) {
          const uint32_t mid = klo + ((khi - klo) >> 1);
          uint32_t cnt = 0;
          for (int r = warp; r < C; r += NVW) cnt += f32_key(tile[r * kFtCols + lane]) <= mid;
          cnt = col_sum_u32(cnt);
          if (cnt > rho) khi = mid; else klo = mid + 1;
        }
        if (bisect) {
          const uint32_t bits = (klo & 0x80000000u) ? (klo & 0x7fffffffu) : ~klo;
          result = __int_as_float((int)bits);
          done = true;
        }
      }
      // gather the (at most 32) candidates of (a, b] per column as row indices, then rank them
      const bool gather = valid && !done;
      const uint32_t m = gather ? cb - ca : 0u;
      if (warp == 0) K->ln[lane] = 0;
      __syncthreads();
      if (gather) {
        for (int i0 = 0; i0 < nrows; i0 += 32) {                          // scan into a mask, then append the few hits
          const float* q = pcol + (size_t)i0 * RSTEP;
          const int n32 = min(32, nrows - i0);
          uint32_t fm = 0u;
          int i = 0;
#pragma unroll 1
          for (; i + 8 <= n32; i += 8, q += 8 * RSTEP) {
            uint32_t h = 0u;
#pragma unroll
            for (int u = 0; u < 8; ++u) {
              const float v = q[u * RSTEP];
              h |= (v > a && v <= bb) ? (1u << u) : 0u;
            }
            fm |= h << i;
          }
          for (; i < n32; ++i, q += RSTEP) {
            const float v = q[0];
            if (v > a && v <= bb) fm |= 1u << i;
          }
          while (fm) {
            const int j = __ffs((int)fm) - 1;
            fm &= fm - 1u;
            K->list[atomicAdd(&K->ln[lane], 1)][lane] = (uint16_t)(warp + NVW * (i0 + j));
          }
        }
      }
      __syncthreads();
      const uint32_t want = rho - ca;
      for (uint32_t i = (uint32_t)warp; i < m; i += NVW) {
        const uint32_t ri = K->list[i][lane];
        const float e = tile[ri * kFtCols + lane];
        uint32_t rank = 0;
        for (uint32_t k2 = 0; k2 < m; ++k2) {
          const uint32_t rk = K->list[k2][lane];
          const float o = tile[rk * kFtCols + lane];
          rank += (o < e) || (o == e && rk < ri);
        }
        if (rank == want) K->med[lane] = e;
      }
      __syncthreads();
      median = gather ? K->med[lane] : result;
      __syncthreads();
    }

    // ------------------------------------------------------------------ F3..F5: thresholds
    float* const gcol = P.dst + (int64_t)y0 * P.stride + s0 + lane;
    for (int it = 0; it < P.n_thr; ++it) {
      const double am = A * rn;
      const double mu = piv + am;
      double var = B * rn - am * am;
      if (!(var > 0.0)) var = 0.0;
      const double cut = P.k[it] * sqrt(var);
      float t_lo, t_hi;
      f32_bounds(mu, cut, t_lo, t_hi);
      const float rv = P.policy == 0 ? (float)mu : median;
      const double dr = (double)rv - piv;
      double dA = 0.0, dB = 0.0;
      uint32_t cnt = 0;
      if (valid) {
        // scan 32 rows at a time into a bit mask (unrolled, compile-time offsets), then visit the few flagged rows
        for (int i0 = 0; i0 < nrows; i0 += 32) {
          const float* q = pcol + (size_t)i0 * RSTEP;
          const int n32 = min(32, nrows - i0);
          uint32_t fm = 0u;
          int i = 0;
#pragma unroll 1
          for (; i + 8 <= n32; i += 8, q += 8 * RSTEP) {
            // eight rows at once through their largest and smallest value (FMNMX3): 2 % of the groups hold a hit at 3 sigma
            float v[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) v[u] = q[u * RSTEP];
            const float mx = fmaxf(fmaxf(fmaxf(v[0], v[1]), fmaxf(v[2], v[3])), fmaxf(fmaxf(v[4], v[5]), fmaxf(v[6], v[7])));
            const float mn = fminf(fminf(fminf(v[0], v[1]), fminf(v[2], v[3])), fminf(fminf(v[4], v[5]), fminf(v[6], v[7])));
            if (mx > t_hi || mn < t_lo) {
              uint32_t h = 0u;
#pragma unroll
              for (int u = 0; u < 8; ++u) h |= (v[u] > t_hi || v[u] < t_lo) ? (1u << u) : 0u;
              fm |= h << i;
            }
          }
          for (; i < n32; ++i, q += RSTEP) {
            const float v = q[0];
            if (v > t_hi || v < t_lo) fm |= 1u << i;
          }
          while (fm) {
            const int j = __ffs((int)fm) - 1;
            fm &= fm - 1u;
            const int r = warp + NVW * (i0 + j);
            const double d = (double)tile[r * kFtCols + lane] - piv;
            dA += dr - d; dB += dr * dr - d * d;
            tile[r * kFtCols + lane] = rv;
            if (!P.copy) gcol[(int64_t)r * P.stride] = rv;
            if (P.flags) P.flags[((int64_t)y0 + r) * P.S + s0 + lane] = 1;
            ++cnt;
          }
        }
      }
      const bool more = it + 1 < P.n_thr;
      if (more || P.counts) {
        const uint32_t total = col_sum_u32(cnt);
        if (P.counts && tid < 32) {                                     // (one copy of every column's total)
          const uint32_t all = __reduce_add_sync(FULL, hwlane < COLS ? total : 0u);
          if (hwlane == 0 && all) atomicAdd(&P.counts[it], (unsigned long long)all);
        }
        if (more && __syncthreads_or(total != 0)) {
          col_sum2(dA, dB);
          const double B_before = B;
          A += dA; B += dB;
          const bool again = valid && total != 0 && (cancels() || B < 1e-6 * B_before);
          if (__syncthreads_or(again)) {
            if (again) piv += A * rn;
            sums(false);
          }
        }
      }
    }

    // ------------------------------------------------------------------ F6: store (out of place), next tile
    fence_proxy_async_smem();                          // generic-proxy accesses of the tile before the async proxy's
    if (P.copy) {
      __syncthreads();
      if (tid == 0) {
        for (int i = 0; i < P.nboxes; ++i)
          ft_tma_store_2d(&maps.dst, s0, y0 + i * P.box_rows, tile + (size_t)i * P.box_rows * kFtCols);
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
