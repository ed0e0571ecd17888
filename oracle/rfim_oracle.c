/*
 * rfim_oracle.c -- CPU ORACLE for the RFIm sigma cuts.  TEST INFRASTRUCTURE ONLY.
 * See rfim_oracle.h for the contract.  Plain C (gcc), single-threaded, no
 * blocking, fusion or reordering beyond what the paper's definition states.
 *
 * Readings of the paper used here (each listed in DESIGN.md, "Readings"):
 *   R1  TDSC statistics are per (beam, channel) time series
 *   R2  sigma is the population standard deviation (divide by N)
 *   R3  the test is strict:  |x - mu| > n sigma
 *   R4  the comparison is two-sided
 *   R5  the replacement mean is the same snapshot mean used in the test
 *       (it includes the outliers)
 *   R6  integer data: replacement mean rounded half up, floor((2S+N)/(2N))
 *   R7  iterations: each threshold sees the data cleaned by the previous one
 *       and recomputes every statistic
 *   R8  flags = OR over iterations; counts[i] = replacements in iteration i
 *   R9  sigma = 0 flags nothing (0 > 0 is false)
 *   R11 windows never overlap or span rows; a short tail is its own window
 *   R12 median = lower median, rank floor((N-1)/2) of the ascending snapshot
 *   R13 the median policy changes the replacement only, not the test
 *   R14 FDSC parameter is the bin SIZE; bins are consecutive channels
 *   R16 FDSC step 2 uses one mean/sigma over all C mean-corrected values
 *   R17 integer data: threshold k quantised to p/2^16, p = round-half-even
 */
#include "rfim_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>

typedef unsigned __int128 u128;
typedef __int128 i128;

#define Q_BITS 16 /* R17: k ~ p / 2^16 */

uint64_t rfim_oracle_quantise_threshold(double k) {
  /* k * 2^16 is exact in binary floating point; nearbyint() rounds half to even
   * in the default rounding mode. */
  return (uint64_t)nearbyint(k * 65536.0);
}

void rfim_oracle_stats_u8(const uint8_t* x, int64_t n, uint64_t* sum, uint64_t* sumsq) {
  uint64_t s = 0, q = 0;
  for (int64_t i = 0; i < n; ++i) {
    s += x[i];
    q += (uint64_t)x[i] * x[i];
  }
  *sum = s;
  *sumsq = q;
}

void rfim_oracle_stats_f32(const float* x, int64_t n, double* mean, double* sigma) {
  /* PAPER.md:100 "the mean (mu), and the standard deviation (sigma)": two plain
   * passes in double, population form (R2). */
  double s = 0.0;
  for (int64_t i = 0; i < n; ++i) s += (double)x[i];
  double mu = s / (double)n;
  double ss = 0.0;
  for (int64_t i = 0; i < n; ++i) {
    double d = (double)x[i] - mu;
    ss += d * d;
  }
  *mean = mu;
  *sigma = sqrt(ss / (double)n);
}

static int cmp_u8(const void* a, const void* b) {
  return (int)*(const uint8_t*)a - (int)*(const uint8_t*)b;
}
static int cmp_f32(const void* a, const void* b) {
  float x = *(const float*)a, y = *(const float*)b;
  return (x > y) - (x < y);
}

/* R12: lower median of a snapshot (the snapshot is copied and sorted). */
static uint8_t lower_median_u8(const uint8_t* x, int64_t n, uint8_t* scratch) {
  memcpy(scratch, x, (size_t)n);
  qsort(scratch, (size_t)n, 1, cmp_u8);
  return scratch[(n - 1) / 2];
}
static float lower_median_f32(const float* x, int64_t n, float* scratch) {
  memcpy(scratch, x, (size_t)n * sizeof(float));
  qsort(scratch, (size_t)n, sizeof(float), cmp_f32);
  return scratch[(n - 1) / 2];
}

/* ------------------------------------------------------------------------- */
/* One sigma-cut iteration on one contiguous series (a TDSC window, or a       */
/* gathered FDSC column with a single bin).  PAPER.md:100.                     */
/* ------------------------------------------------------------------------- */

/* uint8, exact integers.  With S = sum x, Q = sum x^2, V = N Q - S^2 and
 * k = p/q (q = 2^16):   |x - S/N| > k sqrt(V)/N   <=>   q^2 (N x - S)^2 > p^2 V.
 * flag_out[i] receives this iteration's decision; returns the number flagged. */
static uint64_t sigma_cut_iter_u8(uint8_t* x, int64_t n, uint64_t p, int policy,
                                  uint8_t* flag_out, uint8_t* scratch) {
  uint64_t S, Q;
  rfim_oracle_stats_u8(x, n, &S, &Q);                 /* snapshot statistics    */
  u128 V = (u128)n * Q - (u128)S * S;                 /* N^2 * variance, >= 0   */
  u128 rhs = (u128)p * p * V;                         /* p^2 V                  */
  uint8_t r;
  if (policy == RFIM_ORACLE_MEDIAN)
    r = lower_median_u8(x, n, scratch);               /* R12, R13               */
  else
    r = (uint8_t)((2 * S + (uint64_t)n) / (2 * (uint64_t)n)); /* R5, R6         */
  uint64_t nflag = 0;
  for (int64_t i = 0; i < n; ++i) {                   /* decisions from the snapshot */
    i128 d = (i128)n * x[i] - (i128)S;                /* N x - S                */
    u128 lhs = ((u128)(d * d)) << (2 * Q_BITS);       /* q^2 (N x - S)^2        */
    flag_out[i] = (uint8_t)(lhs > rhs);               /* R3 strict, R4 two-sided */
  }
  for (int64_t i = 0; i < n; ++i)                     /* then replace           */
    if (flag_out[i]) { x[i] = r; ++nflag; }
  return nflag;
}

/* float32: statistics and test in double. */
static uint64_t sigma_cut_iter_f32(float* x, int64_t n, double k, int policy,
                                   uint8_t* flag_out, float* scratch) {
  double mu, sigma;
  rfim_oracle_stats_f32(x, n, &mu, &sigma);
  float r = (policy == RFIM_ORACLE_MEDIAN) ? lower_median_f32(x, n, scratch) : (float)mu;
  double cut = k * sigma;
  uint64_t nflag = 0;
  for (int64_t i = 0; i < n; ++i)
    flag_out[i] = (uint8_t)(fabs((double)x[i] - mu) > cut);
  for (int64_t i = 0; i < n; ++i)
    if (flag_out[i]) { x[i] = r; ++nflag; }
  return nflag;
}

/* ------------------------------------------------------------------------- */
/* Argument checks shared by both entry points.                               */
/* ------------------------------------------------------------------------- */
static int check_args(const void* data, int beams, int channels, int samples, int dtype,
                      const double* thresholds, int n_thresholds, int policy,
                      const rfim_oracle_opts* o) {
  if (!data || beams <= 0 || channels <= 0 || samples <= 0) return RFIM_ORACLE_INVALID;
  if (dtype != RFIM_ORACLE_U8 && dtype != RFIM_ORACLE_F32) return RFIM_ORACLE_INVALID;
  if (policy != RFIM_ORACLE_MEAN && policy != RFIM_ORACLE_MEDIAN) return RFIM_ORACLE_INVALID;
  if (n_thresholds < 0 || n_thresholds > 16) return RFIM_ORACLE_INVALID;
  if (n_thresholds > 0 && !thresholds) return RFIM_ORACLE_INVALID;
  for (int i = 0; i < n_thresholds; ++i)
    if (!(thresholds[i] > 0.0) || !(thresholds[i] < 256.0)) return RFIM_ORACLE_INVALID;
  /* integer path: N <= 2^24 keeps every product inside 128 bits */
  if (dtype == RFIM_ORACLE_U8 && (samples > (1 << 24) || channels > (1 << 24)))
    return RFIM_ORACLE_INVALID;
  if (o) {
    if (o->sample_stride != 0 && o->sample_stride < samples) return RFIM_ORACLE_INVALID;
    if (o->window < 0 || o->bin_size < 0) return RFIM_ORACLE_INVALID;
  }
  return RFIM_ORACLE_OK;
}

static size_t elem_size(int dtype) { return dtype == RFIM_ORACLE_U8 ? 1 : 4; }

/* out-of-place: copy every row of data to out, then work on out. */
static void* prepare_output(void* data, int64_t rows, int samples, int64_t stride, int dtype,
                            const rfim_oracle_opts* o) {
  if (!o || !o->out || o->out == data) return data;
  size_t es = elem_size(dtype);
  for (int64_t r = 0; r < rows; ++r)
    memcpy((char*)o->out + (size_t)r * stride * es, (char*)data + (size_t)r * stride * es,
           (size_t)samples * es);
  return o->out;
}

/* ------------------------------------------------------------------------- */
/* TDSC -- PAPER.md:100, Fig. 2                                  */
/* ------------------------------------------------------------------------- */
int rfim_oracle_time_sigma_cut(void* data, int beams, int channels, int samples, int dtype,
                               const double* thresholds, int n_thresholds, int policy,
                               const rfim_oracle_opts* opts) {
  int st = check_args(data, beams, channels, samples, dtype, thresholds, n_thresholds, policy, opts);
  if (st != RFIM_ORACLE_OK) return st;
  int64_t stride = (opts && opts->sample_stride) ? opts->sample_stride : samples;
  int64_t window = (opts && opts->window) ? opts->window : samples;        /* R11 */
  if (window > samples) window = samples;
  int64_t rows = (int64_t)beams * channels;
  void* work = prepare_output(data, rows, samples, stride, dtype, opts);
  uint8_t* flags = opts ? opts->flags : NULL;
  uint64_t* counts = opts ? opts->counts : NULL;
  if (flags) memset(flags, 0, (size_t)rows * samples);
  if (counts) for (int i = 0; i < n_thresholds; ++i) counts[i] = 0;

  uint8_t* iter_flag = (uint8_t*)malloc((size_t)window);
  void* scratch = malloc((size_t)window * 4);
  for (int64_t row = 0; row < rows; ++row) {                 /* R1: rows are independent */
    for (int64_t w0 = 0; w0 < samples; w0 += window) {       /* R11: windows independent */
      int64_t n = (samples - w0 < window) ? samples - w0 : window;
      for (int it = 0; it < n_thresholds; ++it) {            /* R7: sequential           */
        uint64_t nf;
        if (dtype == RFIM_ORACLE_U8) {
          uint8_t* x = (uint8_t*)work + row * stride + w0;
          nf = sigma_cut_iter_u8(x, n, rfim_oracle_quantise_threshold(thresholds[it]), policy,
                                 iter_flag, (uint8_t*)scratch);
        } else {
          float* x = (float*)work + row * stride + w0;
          nf = sigma_cut_iter_f32(x, n, thresholds[it], policy, iter_flag, (float*)scratch);
        }
        if (counts) counts[it] += nf;                        /* R8 */
        if (flags)
          for (int64_t i = 0; i < n; ++i) flags[row * samples + w0 + i] |= iter_flag[i];
      }
    }
  }
  free(iter_flag);
  free(scratch);
  return RFIM_ORACLE_OK;
}

/* ------------------------------------------------------------------------- */
/* FDSC -- PAPER.md:102, Fig. 3                   */
/* ------------------------------------------------------------------------- */

/* One FDSC iteration on one gathered column (C values, one per channel), u8.
 * Step 1: bin means m_b = S_b / n_b; corrected d_c = x_c - m_b(c).
 * Step 2: mean of all d_c is exactly 0 (each bin's corrections sum to 0), so
 *   sigma'^2 = (1/C) sum_c d_c^2 = V / (C n_b),  V = sum_b (n_b Q_b - S_b^2),
 *   and |d_c| > k sigma'  <=>  q^2 C (n_b x_c - S_b)^2 > p^2 n_b V.
 * Flagged ORIGINAL values are replaced by their bin's mean (rounded half up) or
 * lower median. */
static uint64_t fdsc_iter_u8(uint8_t* col, int64_t C, int64_t nb, uint64_t p, int policy,
                             uint8_t* flag_out, uint8_t* scratch, uint64_t* binS, uint8_t* binR) {
  int64_t nbins = C / nb;
  u128 V = 0;
  for (int64_t b = 0; b < nbins; ++b) {
    uint64_t S, Q;
    rfim_oracle_stats_u8(col + b * nb, nb, &S, &Q);
    binS[b] = S;
    V += (u128)nb * Q - (u128)S * S;
    binR[b] = (policy == RFIM_ORACLE_MEDIAN)
                  ? lower_median_u8(col + b * nb, nb, scratch)
                  : (uint8_t)((2 * S + (uint64_t)nb) / (2 * (uint64_t)nb));
  }
  u128 rhs = (u128)p * p * (u128)nb * V;
  uint64_t nflag = 0;
  for (int64_t c = 0; c < C; ++c) {
    i128 d = (i128)nb * col[c] - (i128)binS[c / nb];
    u128 lhs = (((u128)(d * d)) * (u128)C) << (2 * Q_BITS);
    flag_out[c] = (uint8_t)(lhs > rhs);
  }
  for (int64_t c = 0; c < C; ++c)
    if (flag_out[c]) { col[c] = binR[c / nb]; ++nflag; }
  return nflag;
}

/* Same, float32 in double.  Here the paper's steps are followed literally: the
 * mean-corrected values, then THEIR mean and standard deviation (PAPER.md:102
 * "compared to the mean-corrected statistics of all frequency channels"). */
static uint64_t fdsc_iter_f32(float* col, int64_t C, int64_t nb, double k, int policy,
                              uint8_t* flag_out, float* scratch, double* corr, float* binR,
                              double* binM) {
  int64_t nbins = C / nb;
  for (int64_t b = 0; b < nbins; ++b) {
    double s = 0.0;
    for (int64_t j = 0; j < nb; ++j) s += (double)col[b * nb + j];
    binM[b] = s / (double)nb;
    binR[b] = (policy == RFIM_ORACLE_MEDIAN) ? lower_median_f32(col + b * nb, nb, scratch)
                                             : (float)binM[b];
  }
  double s = 0.0;
  for (int64_t c = 0; c < C; ++c) {
    corr[c] = (double)col[c] - binM[c / nb];
    s += corr[c];
  }
  double mu = s / (double)C;
  double ss = 0.0;
  for (int64_t c = 0; c < C; ++c) ss += (corr[c] - mu) * (corr[c] - mu);
  double cut = k * sqrt(ss / (double)C);
  uint64_t nflag = 0;
  for (int64_t c = 0; c < C; ++c) flag_out[c] = (uint8_t)(fabs(corr[c] - mu) > cut);
  for (int64_t c = 0; c < C; ++c)
    if (flag_out[c]) { col[c] = binR[c / nb]; ++nflag; }
  return nflag;
}

int rfim_oracle_freq_sigma_cut(void* data, int beams, int channels, int samples, int dtype,
                               const double* thresholds, int n_thresholds, int policy,
                               const rfim_oracle_opts* opts) {
  int st = check_args(data, beams, channels, samples, dtype, thresholds, n_thresholds, policy, opts);
  if (st != RFIM_ORACLE_OK) return st;
  int64_t stride = (opts && opts->sample_stride) ? opts->sample_stride : samples;
  int64_t nb = (opts && opts->bin_size) ? opts->bin_size : channels;         /* R14 */
  if (nb > channels || channels % nb != 0) return RFIM_ORACLE_INVALID;
  if (nb != channels && nb > 65536) return RFIM_ORACLE_INVALID; /* keeps p^2 n_b V < 2^128 */
  int64_t C = channels;
  int64_t rows = (int64_t)beams * channels;
  void* work = prepare_output(data, rows, samples, stride, dtype, opts);
  uint8_t* flags = opts ? opts->flags : NULL;
  uint64_t* counts = opts ? opts->counts : NULL;
  if (flags) memset(flags, 0, (size_t)rows * samples);
  if (counts) for (int i = 0; i < n_thresholds; ++i) counts[i] = 0;

  size_t es = elem_size(dtype);
  void* col = malloc((size_t)C * es);
  void* scratch = malloc((size_t)C * es);
  uint8_t* iter_flag = (uint8_t*)malloc((size_t)C);
  uint8_t* any_flag = (uint8_t*)malloc((size_t)C);
  uint64_t* binS = (uint64_t*)malloc((size_t)(C / nb) * sizeof(uint64_t));
  double* binM = (double*)malloc((size_t)(C / nb) * sizeof(double));
  void* binR = malloc((size_t)(C / nb) * es);
  double* corr = (double*)malloc((size_t)C * sizeof(double));

  for (int64_t b = 0; b < beams; ++b) {
    for (int64_t s = 0; s < samples; ++s) {                 /* columns are independent */
      for (int64_t c = 0; c < C; ++c) {                     /* gather the column       */
        size_t at = (size_t)((b * C + c) * stride + s);
        if (dtype == RFIM_ORACLE_U8) ((uint8_t*)col)[c] = ((uint8_t*)work)[at];
        else ((float*)col)[c] = ((float*)work)[at];
      }
      memset(any_flag, 0, (size_t)C);
      for (int it = 0; it < n_thresholds; ++it) {
        uint64_t nf;
        if (dtype == RFIM_ORACLE_U8)
          nf = fdsc_iter_u8((uint8_t*)col, C, nb, rfim_oracle_quantise_threshold(thresholds[it]),
                            policy, iter_flag, (uint8_t*)scratch, binS, (uint8_t*)binR);
        else
          nf = fdsc_iter_f32((float*)col, C, nb, thresholds[it], policy, iter_flag,
                             (float*)scratch, corr, (float*)binR, binM);
        if (counts) counts[it] += nf;
        for (int64_t c = 0; c < C; ++c) any_flag[c] |= iter_flag[c];
      }
      for (int64_t c = 0; c < C; ++c) {                     /* scatter back            */
        size_t at = (size_t)((b * C + c) * stride + s);
        if (dtype == RFIM_ORACLE_U8) ((uint8_t*)work)[at] = ((uint8_t*)col)[c];
        else ((float*)work)[at] = ((float*)col)[c];
        if (flags) flags[(size_t)((b * C + c) * samples + s)] = any_flag[c];
      }
    }
  }
  free(col); free(scratch); free(iter_flag); free(any_flag);
  free(binS); free(binM); free(binR); free(corr);
  return RFIM_ORACLE_OK;
}
