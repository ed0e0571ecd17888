/*
 * synth_core.h -- seeded synthetic dynamic spectra (input generator ONLY).
 *
 * This module holds none of the method's arithmetic: it only draws inputs.  It
 * is the one piece of code that both the CUDA path's tests/bench and the CPU
 * oracle's tests are fed from (host twin: synth_host.c, gcc; device twin:
 * synth_cuda.cu, nvcc).  The two twins are bit-identical for uint8 because
 * everything below is integer-only: the Gaussian comes from an inverse-CDF
 * lookup in a table the caller passes in.
 *
 * Value at (beam b, channel c, sample s):
 *   noise(seed, b, c, s)                     counter-based hash -> inverse CDF
 * + row_offset[b][c]                         persistent narrow-band RFI
 * + imp_amp[b][s]                            broadband impulses (all channels)
 * + pulse_amp  if pulse_start[c] <= s < pulse_start[c] + pulse_width   (dispersed pulse, Eq. 2)
 * + sum of burst_amp[j] over the row's bursts j covering s             (intermittent narrow-band RFI)
 * saturated at 255 (uint8) or scaled by 1/f32_scale and added to N(0,1) (float32).
 */
#ifndef RFIM_SYNTH_CORE_H
#define RFIM_SYNTH_CORE_H

#include <stdint.h>

#ifdef __CUDACC__
#define SYNTH_HD __host__ __device__ __forceinline__
#else
#define SYNTH_HD static inline
#endif

typedef struct {
  uint64_t seed;
  int32_t beam0;           /* global index of the first beam in this buffer (enters the hash)   */
  int32_t beams;           /* beams in this buffer                                               */
  int32_t channels;
  int32_t samples;
  int64_t sample_stride;   /* elements between rows of the output buffer                         */
  const uint32_t* cdf;     /* [255] u32: value = #{v : u >= cdf[v]}  (inverse CDF of the noise)  */
  const uint8_t* row_offset;   /* [beams][channels]                                              */
  const uint8_t* imp_amp;      /* [beams][samples]                                               */
  const int32_t* pulse_start;  /* [channels]; pulse disabled when pulse_amp == 0                 */
  int32_t pulse_width;
  int32_t pulse_amp;
  const int32_t* burst_ptr;    /* [beams*channels + 1] CSR offsets into the burst arrays         */
  const int32_t* burst_start;
  const int32_t* burst_len;
  const uint8_t* burst_amp;
  double f32_scale;        /* float32 only: structure amplitudes are divided by this            */
} synth_desc;

/* splitmix64 finaliser (Steele, Lea, Flood 2014), used as a counter-based generator */
SYNTH_HD uint64_t synth_mix64(uint64_t z) {
  z ^= z >> 30; z *= 0xbf58476d1ce4e5b9ULL;
  z ^= z >> 27; z *= 0x94d049bb133111ebULL;
  z ^= z >> 31;
  return z;
}

SYNTH_HD uint64_t synth_hash(uint64_t seed, uint64_t stream, uint64_t row, uint64_t idx) {
  uint64_t h = synth_mix64(seed + 0x9e3779b97f4a7c15ULL * (stream + 1));
  h = synth_mix64(h ^ (row * 0xd1342543de82ef95ULL + 0x632be59bd9b4e019ULL));
  return synth_mix64(h + idx * 0x9e3779b97f4a7c15ULL);
}

/* 32 uniform bits for (global row, sample): two samples share one hash */
SYNTH_HD uint32_t synth_u32(uint64_t seed, uint64_t grow, int64_t s) {
  uint64_t h = synth_hash(seed, 0, grow, (uint64_t)(s >> 1));
  return (s & 1) ? (uint32_t)(h >> 32) : (uint32_t)h;
}

/* inverse CDF: smallest v with u < cdf[v], else 255 */
SYNTH_HD int synth_icdf(const uint32_t* cdf, uint32_t u) {
  int lo = 0, hi = 255;              /* answer in [lo, hi] */
  while (lo < hi) {
    int mid = (lo + hi) >> 1;
    if (u < cdf[mid]) hi = mid; else lo = mid + 1;
  }
  return lo;
}

/* the integer structure (RFI + pulse) added on top of the noise */
SYNTH_HD int synth_structure(const synth_desc* d, int b, int c, int s) {
  int64_t row = (int64_t)b * d->channels + c;
  int v = d->row_offset[row] + d->imp_amp[(int64_t)b * d->samples + s];
  if (d->pulse_amp) {
    int ps = d->pulse_start[c];
    if (s >= ps && s < ps + d->pulse_width) v += d->pulse_amp;
  }
  for (int j = d->burst_ptr[row]; j < d->burst_ptr[row + 1]; ++j)
    if (s >= d->burst_start[j] && s < d->burst_start[j] + d->burst_len[j]) v += d->burst_amp[j];
  return v;
}

SYNTH_HD uint8_t synth_value_u8(const synth_desc* d, int b, int c, int s) {
  uint64_t grow = (uint64_t)(d->beam0 + b) * (uint64_t)d->channels + (uint64_t)c;
  int v = synth_icdf(d->cdf, synth_u32(d->seed, grow, s)) + synth_structure(d, b, c, s);
  return (uint8_t)(v > 255 ? 255 : v);
}

#endif
