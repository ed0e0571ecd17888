// fd_u8.cuh -- frequency-domain sigma cut (FDSC, Fig. 3) for uint8 dynamic spectra, one bin of
// all channels: helpers shared by the FDSC kernels (PRMT transposes, exact per-column byte masks, cluster /
// distributed-shared-memory wrappers used by the strip kernel) and
//   fd_u8_generic_kernel  any pitch / alignment / channel count: one thread per (beam, sample) column,
//       iterations through global memory (L2).  Correctness path for the shapes the fast kernels
//       (fd_u8_quad.cuh, fd_u8_stream.cuh, fd_u8_strip.cuh) do not take; not tuned.
#pragma once

#include "common.cuh"
#include "packed.cuh"

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
};

// ---------------------------------------------------------------- generic kernel
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
