/*
 * rfim_oracle.h -- CPU ORACLE for the RFIm sigma cuts.  TEST INFRASTRUCTURE ONLY.
 *
 * This is the plain, slow, single-threaded restatement of what the paper's two
 * mitigation methods compute (PAPER.md:100 TDSC, PAPER.md:102-108 FDSC,
 * PAPER.md:110 replacement strategy, PAPER.md:142,178 iteration).  It exists so
 * that tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs can check and time the CUDA library against it.  Nothing in
 * the product path (paper_2001_03389_b200/, include/rfim.h, librfim.so) may
 * include, link, import or call anything in this directory, and this directory
 * includes nothing from there: the two share no code.
 *
 * Pinned by tests/test_oracle_pins.py (closed forms, hand-computed arrays,
 * exact rational brute force, numpy library routines, invariants).
 * Unpinned: the paper's accuracy figures (SNR gains, trigger counts,
 * PAPER.md:154-156) -- they need the Crab observation and AMBER, neither of
 * which exists here: "parity unpinned" for those, see DESIGN.md.
 *
 * All pointers are HOST pointers.  Calls are synchronous and single-threaded.
 */
#ifndef RFIM_ORACLE_H
#define RFIM_ORACLE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { RFIM_ORACLE_U8 = 0, RFIM_ORACLE_F32 = 1 };
enum { RFIM_ORACLE_MEAN = 0, RFIM_ORACLE_MEDIAN = 1 };
enum { RFIM_ORACLE_OK = 0, RFIM_ORACLE_INVALID = -1 };

typedef struct {
  int64_t   sample_stride; /* elements between consecutive (beam,channel) rows; 0 = samples */
  int32_t   window;        /* time-domain: statistics window in samples; 0 = whole row      */
  int32_t   bin_size;      /* freq-domain: channels per bin; 0 = one bin of all channels    */
  void*     out;           /* NULL = in place; else same shape/stride as data               */
  uint8_t*  flags;         /* optional dense [B][C][S]; 1 = replaced in any iteration       */
  uint64_t* counts;        /* optional [n_thresholds]; samples replaced in iteration i      */
  void*     reserved;      /* ignored (keeps the argument list parallel to the device ABI)  */
} rfim_oracle_opts;

/* time-domain sigma cut: per (beam, channel) time series (or per
 * window of it), mean and population standard deviation of the current values;
 * samples with |t_i - mu| > n*sigma are replaced by the mean (or the lower
 * median); repeated for each threshold on the already-cleaned data. */
int rfim_oracle_time_sigma_cut(void* data, int beams, int channels, int samples, int dtype,
                               const double* thresholds, int n_thresholds, int policy,
                               const rfim_oracle_opts* opts);

/* frequency-domain sigma cut: per (beam, time sample),
 * channels grouped in bins of bin_size, bin mean subtracted, the mean-corrected
 * values compared with the mean-corrected statistics of all channels; flagged
 * ORIGINAL values replaced by the mean (or lower median) of their bin. */
int rfim_oracle_freq_sigma_cut(void* data, int beams, int channels, int samples, int dtype,
                               const double* thresholds, int n_thresholds, int policy,
                               const rfim_oracle_opts* opts);

/* The integer p with k ~ p / 2^16 that the integer (uint8) tests use
 * (round-half-even of k * 2^16; reading R17). */
uint64_t rfim_oracle_quantise_threshold(double k);

/* Statistics of one contiguous series, exposed so that tests can pin them
 * against numpy / hand-computed values.  u8: exact integers.  f32: fp64. */
void rfim_oracle_stats_u8(const uint8_t* x, int64_t n, uint64_t* sum, uint64_t* sumsq);
void rfim_oracle_stats_f32(const float* x, int64_t n, double* mean, double* sigma);

#ifdef __cplusplus
}
#endif
#endif
