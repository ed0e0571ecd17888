/*
 * synth_host.c -- host twin of the synthetic-input generator (gcc).
 * Input generator only: none of the sigma-cut arithmetic lives here.
 */
#include "synth_core.h"

#include <math.h>

void rfim_synth_fill_u8_host(const synth_desc* d, uint8_t* out) {
  for (int b = 0; b < d->beams; ++b)
    for (int c = 0; c < d->channels; ++c) {
      uint8_t* row = out + ((int64_t)b * d->channels + c) * d->sample_stride;
      for (int s = 0; s < d->samples; ++s) row[s] = synth_value_u8(d, b, c, s);
    }
}

/* float32: N(0,1) by Box-Muller in double from two counter-based uniforms (one
 * pair of normals per pair of samples), plus the integer structure / f32_scale. */
void rfim_synth_fill_f32_host(const synth_desc* d, float* out) {
  const double two_pi = 6.283185307179586476925286766559;
  for (int b = 0; b < d->beams; ++b)
    for (int c = 0; c < d->channels; ++c) {
      uint64_t grow = (uint64_t)(d->beam0 + b) * (uint64_t)d->channels + (uint64_t)c;
      float* row = out + ((int64_t)b * d->channels + c) * d->sample_stride;
      for (int s = 0; s < d->samples; s += 2) {
        uint64_t h1 = synth_hash(d->seed, 1, grow, (uint64_t)(s >> 1));
        uint64_t h2 = synth_hash(d->seed, 2, grow, (uint64_t)(s >> 1));
        double u1 = ((double)(h1 >> 11) + 0.5) * (1.0 / 9007199254740992.0); /* (0,1) */
        double u2 = ((double)(h2 >> 11) + 0.5) * (1.0 / 9007199254740992.0);
        double rad = sqrt(-2.0 * log(u1));
        double g0 = rad * cos(two_pi * u2), g1 = rad * sin(two_pi * u2);
        row[s] = (float)(g0 + (double)synth_structure(d, b, c, s) / d->f32_scale);
        if (s + 1 < d->samples)
          row[s + 1] = (float)(g1 + (double)synth_structure(d, b, c, s + 1) / d->f32_scale);
      }
    }
}
