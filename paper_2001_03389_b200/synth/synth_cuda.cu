/*
 * synth_cuda.cu -- device twin of the synthetic-input generator (nvcc, sm_100a).
 * Input generator only: none of the sigma-cut arithmetic lives here.  All
 * pointers inside the descriptor are DEVICE pointers; `out` is a device pointer.
 * Bit-identical to synth_host.c for uint8 (integer-only).
 */
#include "synth_core.h"

#include <cuda_runtime.h>

__global__ void synth_fill_u8_kernel(synth_desc d, uint8_t* __restrict__ out) {
  __shared__ uint32_t cdf_s[255];
  for (int i = threadIdx.x; i < 255; i += blockDim.x) cdf_s[i] = d.cdf[i];
  __syncthreads();
  d.cdf = cdf_s;
  const int64_t rows = (int64_t)d.beams * d.channels;
  for (int64_t row = blockIdx.x; row < rows; row += gridDim.x) {
    const int b = (int)(row / d.channels), c = (int)(row % d.channels);
    uint8_t* dst = out + row * d.sample_stride;
    for (int s = threadIdx.x; s < d.samples; s += blockDim.x) dst[s] = synth_value_u8(&d, b, c, s);
  }
}

extern "C" int rfim_synth_fill_u8_cuda(const synth_desc* d, uint8_t* out, void* stream) {
  int64_t rows = (int64_t)d->beams * d->channels;
  int grid = (int)(rows < 148 * 16 ? rows : 148 * 16);
  synth_fill_u8_kernel<<<grid, 256, 0, (cudaStream_t)stream>>>(*d, out);
  return (int)cudaGetLastError();
}
