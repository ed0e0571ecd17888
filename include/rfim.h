/*
 * rfim.h -- C ABI of librfim: B200 (sm_100a) sigma-cut RFI cleaning of dynamic spectra.
 *
 * The two mitigation methods of RFIm ("Real-Time RFI Mitigation for the Apertif Radio
 * Transient System", arxiv 2001.03389; citations are PAPER.md line numbers):
 *
 *   rfim_time_sigma_cut   TDSC, PAPER.md:100 (Sec. IV) and Fig. 2:
 *       "For a given frequency channel, each time sample of a batch is compared to the
 *        global statistics of the batch: the mean and the standard deviation.  If t_i is an
 *        outlier (|t_i - mu| > n sigma, n the user-defined threshold) it is replaced by the
 *        mean of the batch."
 *   rfim_freq_sigma_cut   FDSC, PAPER.md:102,108 (Sec. IV) and Fig. 3:
 *       channels at a given time are grouped into bins, the bin mean is subtracted, each
 *       mean-corrected channel is compared to the mean-corrected statistics of all
 *       channels; an outlier's ORIGINAL value is replaced by the mean of its bin.
 *   rfim_time_freq_sigma_cut   both, TDSC then FDSC on its result: the combination the paper
 *       applies to every batch ("combined TDSC=3.25 sigma and FDSC=2.75 sigma").
 *   All take a list of thresholds: the production pipeline iterates ("three iterations
 *   with 3.25 sigma"); iteration i sees the data cleaned by
 *   iteration i-1.  All take a replacement strategy (mean | median).
 *
 * Exact definition (readings of the paper where it is silent: DESIGN.md "Readings"):
 *   population sigma; strict '>'; two-sided; statistics and replacement value are taken
 *   from the snapshot at the start of the iteration; integer data are tested in exact
 *   integer arithmetic with the threshold k quantised to p/2^16 (p = round-half-even):
 *   q^2 (N x - S)^2 > p^2 (N Q - S^2); integer replacement mean = floor((2S+N)/(2N));
 *   median = lower median (rank floor((N-1)/2)); float32 statistics in fp64.
 *
 * Layout: data[beam][channel][sample], sample fastest, rows `sample_stride` elements apart.
 *
 * Ownership / execution: every data pointer of the device entry points is a DEVICE pointer
 * owned by the caller; the library allocates no device memory for them.  The `thresholds`
 * arrays are HOST memory, read before the call returns.  Work is enqueued on `opts->stream`
 * and the call returns without synchronising; no host read of device memory.  The library
 * keeps no data between calls; it caches per-process launch attributes (shared-memory
 * limits, occupancy) and the last tensor-map encodings, keyed on pointer and shape.
 * `out` must be `data` itself (or NULL) or must not overlap it.
 *
 * Errors: return value only (no exceptions, errno or abort).  RFIM_ERR_INVALID and
 * RFIM_ERR_UNSUPPORTED are decided before anything is enqueued.  RFIM_ERR_CUDA (a failed
 * memset, copy or launch) leaves the outputs undefined: earlier operations of the same call
 * may already be queued.  There is no CPU fallback: a missing device is RFIM_ERR_CUDA.
 *
 * Reads around the data: the uint8 FDSC kernels fetch row segments through TMA tensor maps / bulk copies, whose
 * granule is 16 bytes: up to 15 bytes before a row segment and after it (inside the same 16-byte aligned granule,
 * hence inside the same page) are READ and ignored -- also the bytes just before `data` (with bins: and `out`) and
 * just behind the last row when those are not 16-byte aligned.  Nothing outside the samples is ever written.
 *
 * Performance notes (DESIGN.md section 6 and BASELINE.md section 4 have the numbers).  Tuned kernels exist for:
 *   uint8 TDSC on whole rows of <= 65000 samples, mean or median;
 *   uint8 FDSC, one bin, mean (any channel count that is a multiple of 4) or median (tiles that fit one CTA: up
 *     to about 1570 channels); 512 / 1024 / 1536 / 2048 channels with mean replacement take a streaming kernel on
 *     large in-place batches, and also accept bins whose size is a multiple of 16, at most 256, and divides
 *     channels / 2 (a kernel that streams the data once per threshold plus once; out of place it reads `out` back
 *     through tensor maps of its own, with the same 16-byte granule as described above);
 *   float32 TDSC on rows that fit shared memory (<= about 56000 samples) with windows that are multiples of 4
 *     samples (or the whole row), 16-byte aligned rows, mean or median;
 *   float32 FDSC, one bin or bins of at most 64 channels, mean or median, 16-byte aligned rows, channels x 128
 *     bytes <= about 220 KB.
 * Everything else the ABI accepts (uint8 TDSC with windows or rows longer than 65000 samples, uint8 FDSC with median
 * replacement and bins, or odd bin sizes, float32 FDSC with bins of more than 64 channels, unaligned float32 rows)
 * runs in definition kernels (one thread per column / one CTA per row) that go through L2 several times: 10 to 50
 * times slower.
 */
#ifndef RFIM_H
#define RFIM_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define RFIM_VERSION 200 /* 0.2.0 */
#define RFIM_MAX_THRESHOLDS 16

typedef enum { RFIM_U8 = 0, RFIM_F32 = 1 } rfim_dtype;
typedef enum { RFIM_REPLACE_MEAN = 0, RFIM_REPLACE_MEDIAN = 1 } rfim_replace;

enum {
  RFIM_OK = 0,
  RFIM_ERR_INVALID = -1,     /* bad argument (list below)                                  */
  RFIM_ERR_UNSUPPORTED = -2, /* valid request that no kernel (of the forced variant) runs  */
  RFIM_ERR_CUDA = -3,        /* CUDA runtime error (text: rfim_last_cuda_error)            */
  RFIM_ERR_TOO_LARGE = -4    /* rfim_freq_sigma_cut_noalloc: beyond RFIM_NOALLOC_MAX_TILES */
};

/* rfim_workspace_bytes `op` */
enum { RFIM_OP_TIME = 0, RFIM_OP_FREQ = 1, RFIM_OP_TIME_FREQ = 2, RFIM_OP_HOST = 3 };

typedef struct {
  int64_t   sample_stride; /* elements between consecutive (beam,channel) rows; 0 = samples (dense) */
  int32_t   window;        /* time-domain only: statistics window in samples; 0 = whole row         */
  int32_t   bin_size;      /* freq-domain only: channels per bin; 0 = one bin of all channels       */
  void*     out;           /* device; NULL = in place; else same shape/stride as data (may == data) */
  uint8_t*  flags;         /* device, optional dense [B][C][S]; 1 = replaced in ANY iteration, else 0 */
  uint64_t* counts;        /* device, optional [n_thresholds]; samples replaced in iteration i
                              (overwritten, not accumulated; a sample can be counted twice);
                              rfim_time_freq_sigma_cut: [n_time + n_freq], time iterations first    */
  void*     stream;        /* cudaStream_t; NULL = legacy default stream                            */
  void*     workspace;     /* device scratch of >= rfim_workspace_bytes(...) bytes, or NULL        */
  int32_t   variant;       /* 0 = auto.  Non-zero selects a kernel variant (testing / tuning):
                              1 = generic correctness kernels, 2 = a tuned kernel or RFIM_ERR_UNSUPPORTED;
                              TDSC only: 3 / 4 = staged kernel with one / two warps per row;
                              FDSC only: 13 = strip kernel with per-row bulk copies, 14 = strip kernel in
                              clusters (never the whole tile in one CTA), 15 = strip kernel, 16 = streaming
                              kernel (one bin or bins), 17 = streaming kernel with one warp per alignment
                              class (one bin), 18 = the same with the per-bin mean correction (bins).
                              A variant that cannot run the request, or belongs to the other
                              operation, returns RFIM_ERR_UNSUPPORTED.                              */
  int32_t   reserved;      /* must be 0                                                            */
} rfim_opts;               /* opts == NULL means all zeros                                          */

/*
 * Time-domain sigma cut (TDSC) -- PAPER.md:100, Fig. 2.
 *   data        device pointer, [beams][channels][samples] of `dtype`, rows sample_stride apart
 *   thresholds  host array of n_thresholds sigma multiples, applied in order (0 <= n <= 16)
 *   policy      replacement value: snapshot mean or lower median
 *   opts->window  statistics are per non-overlapping window of this many samples within a row
 *                 (the last window of a row may be shorter); 0 = the whole row (the paper's batch)
 * RFIM_ERR_INVALID: NULL data; a dimension <= 0; n_thresholds outside [0,16]; NULL thresholds with
 *   n > 0; a threshold that is NaN, <= 0 or >= 256; sample_stride in (0, samples); window < 0;
 *   bin_size < 0; unknown enum or variant; RFIM_U8 with samples > 2^24; reserved != 0; flags/counts/out
 *   misaligned for their type; out overlapping data without being data.
 * n_thresholds == 0 is a valid no-op (copies data to out when out-of-place).
 */
int rfim_time_sigma_cut(void* data, int beams, int channels, int samples, rfim_dtype dtype,
                        const double* thresholds, int n_thresholds, rfim_replace policy,
                        const rfim_opts* opts);

/*
 * Frequency-domain sigma cut (FDSC) -- PAPER.md:102,108, Fig. 3.
 *   As above, statistics across the `channels` axis for every (beam, sample).
 *   opts->bin_size  channels per bin for step 1 (bin-mean correction); must divide channels;
 *                   0 = one bin of all channels (then FDSC is TDSC along the channel axis).
 * In place, a sample that is not replaced is not rewritten.
 * Additional RFIM_ERR_INVALID: bin_size not dividing channels; RFIM_U8 with channels > 2^24 or
 *   1 < bin_size < channels with bin_size > 65536.
 */
int rfim_freq_sigma_cut(void* data, int beams, int channels, int samples, rfim_dtype dtype,
                        const double* thresholds, int n_thresholds, rfim_replace policy,
                        const rfim_opts* opts);

/*
 * FDSC without any device allocation -- the same operation for callers that cannot call
 * cudaMalloc: code under CUDA graph capture, tight serving loops, harnesses that forbid allocation.  Same
 * arguments and results as rfim_freq_sigma_cut, restricted to what the streaming kernel covers: RFIM_U8,
 * RFIM_REPLACE_MEAN, one bin (bin_size 0 or channels), channels in {512, 1024, 1536, 2048}, rows 4-byte aligned
 * (data, out and the stride multiples of 4) -- anything else is RFIM_ERR_UNSUPPORTED -- and at most
 * RFIM_NOALLOC_MAX_TILES tiles per call, a tile being 128 samples of one beam:
 *     beams * ceil(samples / 128) <= RFIM_NOALLOC_MAX_TILES, else RFIM_ERR_TOO_LARGE (nothing is enqueued).
 * opts->workspace must be NULL and opts->variant 0 (RFIM_ERR_INVALID otherwise): the kernel's scratch, its tile
 * dispenser, is a static device array of RFIM_NOALLOC_SCRATCH_BYTES bytes inside the library, held by every GPU
 * that loads the library until the process exits.  The call makes no cudaMalloc / cudaFree / cudaMallocAsync or
 * other allocating call; it enqueues one 4-byte memset of the dispenser, the clearing of flags / counts if given,
 * and the kernel on opts->stream.  The first call on a device also looks up the array's device address and the
 * kernel's launch attributes: make it once outside a stream capture.
 * All calls on a device share the array: calls that follow one another on a stream are fine, calls that OVERLAP
 * on the GPU (different streams without a dependency between them) race on the dispenser and give wrong results.
 */
#define RFIM_NOALLOC_SCRATCH_BYTES 256
#define RFIM_NOALLOC_MAX_TILES (1 << 24)
int rfim_freq_sigma_cut_noalloc(void* data, int beams, int channels, int samples, rfim_dtype dtype,
                                const double* thresholds, int n_thresholds, rfim_replace policy,
                                const rfim_opts* opts);

/*
 * TDSC followed by FDSC on its result -- PAPER.md:118,144.  Equivalent to rfim_time_sigma_cut(data -> out)
 * followed by rfim_freq_sigma_cut(out, in place), on the same stream: TDSC reads `data` and writes `out` (or
 * works in place), FDSC then cleans that result in place.  opts->window applies to TDSC, opts->bin_size to
 * FDSC; flags = replaced by either; counts = [n_time + n_freq].  Either list may be empty.
 */
int rfim_time_freq_sigma_cut(void* data, int beams, int channels, int samples, rfim_dtype dtype,
                             const double* time_thresholds, int n_time,
                             const double* freq_thresholds, int n_freq,
                             rfim_replace policy, const rfim_opts* opts);

/*
 * Host-buffer convenience (end-to-end path): `data` and `out` are HOST pointers (pinned memory
 * gives full PCIe rate; pageable works).  Beams are streamed in chunks through three device staging
 * buffers: H2D copy, rfim_time_freq_sigma_cut on the chunk, D2H copy, overlapped across chunks on three
 * internal streams.  The staging buffers are taken from opts->workspace (device memory of at least
 * rfim_workspace_bytes(RFIM_OP_HOST, ...) bytes); with workspace == NULL the call allocates and frees
 * them itself (slower: a cudaMalloc / cudaFree pair per call).  Synchronous: returns when `out` (or
 * `data`, if out is NULL) holds the result.  opts->out / flags / counts / stream must be NULL here;
 * sample_stride, window, bin_size, workspace apply.  Only the operations that run (n_time > 0, n_freq > 0)
 * are validated.  On RFIM_ERR_CUDA `out` may be partly written.
 */
int rfim_sigma_cut_host(void* data, void* out, int beams, int channels, int samples, rfim_dtype dtype,
                        const double* time_thresholds, int n_time,
                        const double* freq_thresholds, int n_freq,
                        rfim_replace policy, const rfim_opts* opts);

/* Bytes of device scratch the given call uses from opts->workspace (0 = none).  `op`: RFIM_OP_*.  The device
 * entry points need none today; RFIM_OP_HOST returns the size of the three staging buffers. */
size_t rfim_workspace_bytes(int op, int beams, int channels, int samples, rfim_dtype dtype,
                            int n_thresholds, rfim_replace policy, const rfim_opts* opts);

/* Number of kernel launches the library has enqueued in this process (for bench accounting). */
uint64_t rfim_launch_count(void);

/* Name of the kernel variant the last successful call on this thread selected ("" before any). */
const char* rfim_last_variant(void);

const char* rfim_status_string(int status);
const char* rfim_last_cuda_error(void); /* text of the last RFIM_ERR_CUDA on this thread */
int         rfim_version(void);

#ifdef __cplusplus
}
#endif
#endif /* RFIM_H */
