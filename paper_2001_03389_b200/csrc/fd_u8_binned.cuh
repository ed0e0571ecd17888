// fd_u8_binned.cuh -- frequency-domain sigma cut with the paper's step 1, the per-bin mean correction
// (Fig. 5 uses bins of 32 channels), for uint8 dynamic spectra.
// SURVEY.md 8f NEXT-1.  Correctness path: one thread per (beam, sample) column, all passes through L2.
//
// Per time sample and iteration, with bins of nb consecutive channels (readings R14..R16):
//   S_b, Q_b = sum, sum of squares of bin b;   corrected value d_c = x_c - S_b/nb;   the mean of all corrected
//   values is exactly 0, so sigma'^2 = V / (C nb) with V = sum_b (nb Q_b - S_b^2), and
//   |d_c| > k sigma'  <=>  2^32 C (nb x_c - S_b)^2 > p^2 nb V  <=>  (nb x_c - S_b)^2 > floor(p^2 nb V / (2^32 C)) =: W.
//   A flagged ORIGINAL value is replaced by its bin's mean, rounded half up: floor((2 S_b + nb) / (2 nb)).
// Every decision of an iteration uses the snapshot V; a bin's S_b is read before the bin is modified.
#pragma once

#include "common.cuh"

namespace rfim {

struct FdBinnedParams {
  const uint8_t* src;
  uint8_t* dst;
  int64_t stride;
  int beams, C, S, nb;
  int n_thr;
  int policy;                   // 0 = bin mean (rounded half up), 1 = lower median of the bin
  uint32_t p[16];
  uint8_t* flags;
  unsigned long long* counts;
};

constexpr int kFdBinnedThreads = 128;

__global__ void __launch_bounds__(kFdBinnedThreads) fd_u8_binned_kernel(const FdBinnedParams P) {
  typedef unsigned __int128 u128;
  const int64_t ncol = (int64_t)P.beams * P.S;
  const int nbins = P.C / P.nb;
  for (int64_t col = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; col < ncol;
       col += (int64_t)gridDim.x * blockDim.x) {
    const int b = (int)(col / P.S), s = (int)(col % P.S);
    const uint8_t* src = P.src + (int64_t)b * P.C * P.stride + s;
    uint8_t* dst = P.dst + (int64_t)b * P.C * P.stride + s;
    if (dst != src)
      for (int c = 0; c < P.C; ++c) dst[(int64_t)c * P.stride] = src[(int64_t)c * P.stride];
    for (int it = 0; it < P.n_thr; ++it) {
      // snapshot: V over all bins
      uint64_t V = 0;
      for (int bin = 0; bin < nbins; ++bin) {
        uint64_t Sb = 0, Qb = 0;
        for (int j = 0; j < P.nb; ++j) {
          const uint32_t x = dst[(int64_t)(bin * P.nb + j) * P.stride];
          Sb += x; Qb += x * x;
        }
        V += (uint64_t)P.nb * Qb - Sb * Sb;
      }
      const u128 rhs = (u128)((uint64_t)P.p[it] * P.p[it]) * ((u128)(uint64_t)P.nb * V);   // p^2 nb V < 2^120
      const u128 Wfull = (rhs >> 32) / (u128)(uint64_t)P.C;   // floor(floor(rhs / 2^32) / C) = floor(rhs / (2^32 C))
      const bool never = (Wfull >> 64) != 0;
      const uint64_t W = (uint64_t)Wfull;
      uint32_t cnt = 0;
      if (!never) {
        for (int bin = 0; bin < nbins; ++bin) {
          uint64_t Sb = 0;
          for (int j = 0; j < P.nb; ++j) Sb += dst[(int64_t)(bin * P.nb + j) * P.stride];
          uint32_t r = (uint32_t)((2 * Sb + (uint64_t)P.nb) / (2 * (uint64_t)P.nb));
          if (P.policy == 1) {
            // lower median (rank (nb - 1) / 2) of the bin's snapshot: smallest v with #{x <= v} > rank, by
            // bisection on the byte value with counting passes (8 passes; correctness path)
            const uint32_t rank = (uint32_t)(P.nb - 1) >> 1;
            uint32_t lo_v = 0, hi_v = 255;
            while (lo_v < hi_v) {
              const uint32_t mid = (lo_v + hi_v) >> 1;
              uint32_t le = 0;
              for (int j = 0; j < P.nb; ++j) le += dst[(int64_t)(bin * P.nb + j) * P.stride] <= mid;
              if (le > rank) hi_v = mid; else lo_v = mid + 1;
            }
            r = lo_v;
          }
          for (int j = 0; j < P.nb; ++j) {
            const int c = bin * P.nb + j;
            const uint32_t x = dst[(int64_t)c * P.stride];
            const int64_t d = (int64_t)((uint64_t)P.nb * x) - (int64_t)Sb;     // |d| < 2^24
            if ((uint64_t)(d * d) > W) {
              dst[(int64_t)c * P.stride] = (uint8_t)r;
              ++cnt;
              if (P.flags) P.flags[((int64_t)b * P.C + c) * P.S + s] = 1;
            }
          }
        }
      }
      if (cnt && P.counts) atomicAdd(&P.counts[it], (unsigned long long)cnt);
    }
  }
}

}  // namespace rfim
