// fd_f32.cuh -- frequency-domain sigma cut (FDSC) for float32 dynamic spectra: bins,
// mean or lower-median replacement.  SURVEY.md 8f NEXT-3.  Correctness path: one thread per (beam, sample)
// column, fp64 arithmetic in the order of the definition (bin means, mean-corrected values, THEIR mean and
// population standard deviation, strict two-sided test, flagged ORIGINAL values replaced by the bin's mean or
// lower median), every pass through L2.  Statistics and replacement values come from the snapshot at the start
// of the iteration: a bin's mean / median is taken before the bin is modified, and mu', sigma' before any bin is.
#pragma once

#include "common.cuh"
#include "td_f32.cuh"   // f32_key

namespace rfim {

struct FdF32Params {
  const float* src;
  float* dst;
  int64_t stride;
  int beams, C, S, nb;
  int n_thr;
  int policy;
  double k[16];
  uint8_t* flags;
  unsigned long long* counts;
};

constexpr int kFdF32Threads = 128;

__device__ __forceinline__ double fd_f32_bin_mean(const float* col, int64_t stride, int c0, int nb) {
  double s = 0.0;
  for (int j = 0; j < nb; ++j) s += (double)col[(int64_t)(c0 + j) * stride];
  return s / (double)nb;
}

// lower median of the nb values of one bin: bisection on the order-preserving keys with counting passes
__device__ __forceinline__ float fd_f32_bin_median(const float* col, int64_t stride, int c0, int nb) {
  const uint32_t rank = (uint32_t)(nb - 1) >> 1;
  uint32_t klo = 0u, khi = 0xffffffffu;
  while (klo < khi) {
    const uint32_t mid = klo + ((khi - klo) >> 1);
    uint32_t le = 0;
    for (int j = 0; j < nb; ++j) le += f32_key(col[(int64_t)(c0 + j) * stride]) <= mid;
    if (le > rank) khi = mid; else klo = mid + 1;
  }
  // return the ELEMENT with that key (keeps the sign of a zero as stored)
  for (int j = 0; j < nb; ++j) {
    const float v = col[(int64_t)(c0 + j) * stride];
    if (f32_key(v) == klo) return v;
  }
  return 0.0f;
}

__global__ void __launch_bounds__(kFdF32Threads) fd_f32_generic_kernel(const FdF32Params P) {
  const int64_t ncol = (int64_t)P.beams * P.S;
  const int nbins = P.C / P.nb;
  for (int64_t col = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; col < ncol;
       col += (int64_t)gridDim.x * blockDim.x) {
    const int b = (int)(col / P.S), s = (int)(col % P.S);
    const float* src = P.src + (int64_t)b * P.C * P.stride + s;
    float* dst = P.dst + (int64_t)b * P.C * P.stride + s;
    if (dst != src)
      for (int c = 0; c < P.C; ++c) dst[(int64_t)c * P.stride] = src[(int64_t)c * P.stride];
    for (int it = 0; it < P.n_thr; ++it) {
      // snapshot statistics of the mean-corrected values
      double sum = 0.0;
      for (int bin = 0; bin < nbins; ++bin) {
        const double m = fd_f32_bin_mean(dst, P.stride, bin * P.nb, P.nb);
        for (int j = 0; j < P.nb; ++j) sum += (double)dst[(int64_t)(bin * P.nb + j) * P.stride] - m;
      }
      const double mu = sum / (double)P.C;
      double ss = 0.0;
      for (int bin = 0; bin < nbins; ++bin) {
        const double m = fd_f32_bin_mean(dst, P.stride, bin * P.nb, P.nb);
        for (int j = 0; j < P.nb; ++j) {
          const double d = ((double)dst[(int64_t)(bin * P.nb + j) * P.stride] - m) - mu;
          ss += d * d;
        }
      }
      const double cut = P.k[it] * sqrt(ss / (double)P.C);
      uint32_t cnt = 0;
      for (int bin = 0; bin < nbins; ++bin) {
        const double m = fd_f32_bin_mean(dst, P.stride, bin * P.nb, P.nb);     // before the bin is modified
        const float r = P.policy == 1 ? fd_f32_bin_median(dst, P.stride, bin * P.nb, P.nb) : (float)m;
        for (int j = 0; j < P.nb; ++j) {
          const int c = bin * P.nb + j;
          const double d = ((double)dst[(int64_t)c * P.stride] - m) - mu;
          if (fabs(d) > cut) {
            dst[(int64_t)c * P.stride] = r;
            ++cnt;
            if (P.flags) P.flags[((int64_t)b * P.C + c) * P.S + s] = 1;
          }
        }
      }
      if (cnt && P.counts) atomicAdd(&P.counts[it], (unsigned long long)cnt);
    }
  }
}

}  // namespace rfim
