// rfim_api.cu -- the C ABI of librfim (include/rfim.h): argument checks, the order of operations, the host path.
// No CPU fallback: every step of the path runs in the kernels of this directory (launch_*.cu).
#include "host.h"

#include <cmath>
#include <cstdio>

namespace rfim_host {
uint64_t launches();
const char* last_variant();
const char* last_cuda_error();
}  // namespace rfim_host

using namespace rfim_host;

namespace {

// op: 0 time, 1 freq
int validate(int op, void* data, int beams, int channels, int samples, rfim_dtype dtype,
             const double* thr, int n_thr, rfim_replace policy, const rfim_opts* o, Call& c) {
  if (!data || beams <= 0 || channels <= 0 || samples <= 0) return RFIM_ERR_INVALID;
  if (dtype != RFIM_U8 && dtype != RFIM_F32) return RFIM_ERR_INVALID;
  if (policy != RFIM_REPLACE_MEAN && policy != RFIM_REPLACE_MEDIAN) return RFIM_ERR_INVALID;
  if (n_thr < 0 || n_thr > RFIM_MAX_THRESHOLDS) return RFIM_ERR_INVALID;
  if (n_thr > 0 && !thr) return RFIM_ERR_INVALID;
  for (int i = 0; i < n_thr; ++i)
    if (!(thr[i] > 0.0) || !(thr[i] < 256.0)) return RFIM_ERR_INVALID;   // also rejects NaN
  if (dtype == RFIM_U8 && (op == 0 ? samples : channels) > (1 << 24)) return RFIM_ERR_INVALID;
  rfim_opts z;
  memset(&z, 0, sizeof(z));
  if (o) z = *o;
  if (z.reserved != 0) return RFIM_ERR_INVALID;
  if (z.sample_stride != 0 && z.sample_stride < samples) return RFIM_ERR_INVALID;
  if (z.window < 0 || z.bin_size < 0) return RFIM_ERR_INVALID;
  if (z.variant < 0 || z.variant > 18 || (z.variant >= 5 && z.variant <= 12)) return RFIM_ERR_INVALID;
  if (op == 1 && z.bin_size != 0) {
    if (z.bin_size > channels || channels % z.bin_size != 0) return RFIM_ERR_INVALID;
    if (dtype == RFIM_U8 && z.bin_size != channels && z.bin_size > 65536) return RFIM_ERR_INVALID;
  }
  const size_t es = elem_size(dtype);
  if ((reinterpret_cast<uintptr_t>(data) % es) != 0) return RFIM_ERR_INVALID;
  if (z.out && (reinterpret_cast<uintptr_t>(z.out) % es) != 0) return RFIM_ERR_INVALID;
  if (z.counts && (reinterpret_cast<uintptr_t>(z.counts) % 8) != 0) return RFIM_ERR_INVALID;
  c.data = data;
  c.out = z.out ? z.out : data;
  c.beams = beams; c.channels = channels; c.samples = samples;
  c.dtype = dtype; c.thr = thr; c.n_thr = n_thr; c.policy = policy;
  c.stride = z.sample_stride ? z.sample_stride : samples;
  c.window = (z.window == 0 || z.window > samples) ? samples : z.window;
  c.bin_size = (z.bin_size == 0) ? channels : z.bin_size;
  c.flags = z.flags;
  c.counts = reinterpret_cast<unsigned long long*>(z.counts);
  c.stream = reinterpret_cast<cudaStream_t>(z.stream);
  c.workspace = z.workspace;
  if (z.workspace && (reinterpret_cast<uintptr_t>(z.workspace) & 255) != 0) return RFIM_ERR_INVALID;
  c.variant = z.variant;
  c.reserved_team = 0;
  c.keep_outputs = false;
  if (c.out != c.data) {                   // out of place: the two buffers must not overlap
    const uintptr_t a = reinterpret_cast<uintptr_t>(c.data), b = reinterpret_cast<uintptr_t>(c.out);
    const uintptr_t extent = (uintptr_t)(((size_t)beams * channels - 1) * (size_t)c.stride + samples) * es;
    if (a < b + extent && b < a + extent) return RFIM_ERR_INVALID;
  }
  if (op == 0) {
    if (z.variant >= 13) return RFIM_ERR_UNSUPPORTED;               // FDSC-only variants
    if (z.variant == 3 || z.variant == 4) { c.reserved_team = z.variant - 2; c.variant = 2; }
  } else {
    if (z.variant == 3 || z.variant == 4) return RFIM_ERR_UNSUPPORTED;   // TDSC-only variants
  }
  return RFIM_OK;
}

int copy_through(const Call& c) {   // n_thresholds == 0, out of place
  if (c.out != c.data) {
    const size_t es = elem_size(c.dtype);
    CUDA_TRY(cudaMemcpy2DAsync(c.out, (size_t)c.stride * es, c.data, (size_t)c.stride * es,
                               (size_t)c.samples * es, (size_t)c.beams * c.channels,
                               cudaMemcpyDeviceToDevice, c.stream));
  }
  return RFIM_OK;
}

int run_time(const Call& c) {
  if (c.n_thr == 0) {
    int st = clear_outputs(c);
    if (st != RFIM_OK) return st;
    return copy_through(c);
  }
  return c.dtype == RFIM_U8 ? launch_td_u8(c) : launch_td_f32(c);
}
int run_freq(const Call& c) {
  if (c.n_thr == 0) {
    int st = clear_outputs(c);
    if (st != RFIM_OK) return st;
    return copy_through(c);
  }
  return c.dtype == RFIM_U8 ? launch_fd_u8(c) : launch_fd_f32(c);
}

// TDSC (data -> out) then FDSC (out, in place) on one stream; ct / cf were validated by the caller
int run_time_freq(Call ct, Call cf) {
  // flags = replaced by either operation, counts = [n_time + n_freq]: prepared once, then both kernels add to them
  Call both = ct;
  both.n_thr = ct.n_thr + cf.n_thr;
  both.keep_outputs = false;
  int st = clear_outputs(both);
  if (st != RFIM_OK) return st;
  ct.keep_outputs = true;
  cf.keep_outputs = true;
  cf.data = ct.out;
  cf.out = ct.out;
  if (cf.counts) cf.counts += ct.n_thr;
  if (ct.n_thr > 0 || ct.out != ct.data) {
    if ((st = run_time(ct)) != RFIM_OK) return st;
  }
  if (cf.n_thr > 0) {
    if ((st = run_freq(cf)) != RFIM_OK) return st;
  }
  return RFIM_OK;
}

// geometry of the host path: chunks of whole beams, about 128 MiB (long enough copies for full PCIe rate, short
// enough to overlap three of them)
constexpr int kHostSlots = 3;
int host_chunk_beams(int beams, int channels, int64_t stride, size_t es) {
  const size_t beam_bytes = (size_t)channels * (size_t)stride * es;
  int per_chunk = (int)((size_t)(128u << 20) / beam_bytes);
  if (per_chunk < 1) per_chunk = 1;
  if (per_chunk > beams) per_chunk = beams;
  return per_chunk;
}

struct HostStreams {
  cudaStream_t s[kHostSlots] = {nullptr, nullptr, nullptr};
  int dev = -1;
};
// three internal streams per host thread, created on first use (stream creation is slow enough to show up in a
// 9 GB end-to-end call otherwise); they hold no data
int host_streams(HostStreams*& out) {
  thread_local HostStreams hs;
  int dev = 0;
  int st = current_device(dev);
  if (st != RFIM_OK) return st;
  if (hs.dev != dev) {
    for (int i = 0; i < kHostSlots; ++i) {
      if (hs.s[i]) cudaStreamDestroy(hs.s[i]);
      hs.s[i] = nullptr;
      CUDA_TRY(cudaStreamCreateWithFlags(&hs.s[i], cudaStreamNonBlocking));
    }
    hs.dev = dev;
  }
  out = &hs;
  return RFIM_OK;
}

}  // namespace

// =============================================================================================
extern "C" {

int rfim_time_sigma_cut(void* data, int beams, int channels, int samples, rfim_dtype dtype,
                        const double* thresholds, int n_thresholds, rfim_replace policy,
                        const rfim_opts* opts) {
  Call c;
  int st = validate(0, data, beams, channels, samples, dtype, thresholds, n_thresholds, policy, opts, c);
  if (st != RFIM_OK) return st;
  return run_time(c);
}

int rfim_freq_sigma_cut(void* data, int beams, int channels, int samples, rfim_dtype dtype,
                        const double* thresholds, int n_thresholds, rfim_replace policy,
                        const rfim_opts* opts) {
  Call c;
  int st = validate(1, data, beams, channels, samples, dtype, thresholds, n_thresholds, policy, opts, c);
  if (st != RFIM_OK) return st;
  return run_freq(c);
}

int rfim_time_freq_sigma_cut(void* data, int beams, int channels, int samples, rfim_dtype dtype,
                             const double* time_thresholds, int n_time,
                             const double* freq_thresholds, int n_freq,
                             rfim_replace policy, const rfim_opts* opts) {
  if (n_time < 0 || n_time > RFIM_MAX_THRESHOLDS || n_freq < 0 || n_freq > RFIM_MAX_THRESHOLDS) return RFIM_ERR_INVALID;
  rfim_opts o;
  memset(&o, 0, sizeof(o));
  if (opts) o = *opts;
  // variants 0 (auto), 1 (generic kernels) and 2 (tuned kernels) apply to both operations; the others belong to one
  const int variant = o.variant;
  if (variant > 2) o.variant = 0;
  Call ct, cf;
  int st = validate(0, data, beams, channels, samples, dtype, time_thresholds, n_time, policy, &o, ct);
  if (st != RFIM_OK) return st;
  st = validate(1, data, beams, channels, samples, dtype, freq_thresholds, n_freq, policy, &o, cf);
  if (st != RFIM_OK) return st;
  if (variant > 18 || (variant >= 5 && variant <= 12)) return RFIM_ERR_INVALID;
  if (variant > 2) return RFIM_ERR_UNSUPPORTED;
  return run_time_freq(ct, cf);
}

int rfim_sigma_cut_host(void* data, void* out, int beams, int channels, int samples, rfim_dtype dtype,
                        const double* time_thresholds, int n_time,
                        const double* freq_thresholds, int n_freq,
                        rfim_replace policy, const rfim_opts* opts) {
  if (opts && (opts->out || opts->flags || opts->counts || opts->stream)) return RFIM_ERR_INVALID;
  if (n_time < 0 || n_time > RFIM_MAX_THRESHOLDS || n_freq < 0 || n_freq > RFIM_MAX_THRESHOLDS) return RFIM_ERR_INVALID;
  // validate exactly as the device entry points do (the host pointers are never dereferenced here); an operation
  // that does not run (no thresholds) is only checked for the arguments both share
  rfim_opts o;
  memset(&o, 0, sizeof(o));
  if (opts) { o.sample_stride = opts->sample_stride; o.window = opts->window; o.bin_size = opts->bin_size; o.reserved = opts->reserved; }
  void* const workspace = opts ? opts->workspace : nullptr;
  Call ct, cf;
  rfim_opts ot = o, of = o;
  if (n_freq == 0) ot.bin_size = 0;
  if (n_time == 0) of.window = 0;
  if (n_freq == 0) of.bin_size = 0;
  int st = validate(0, data, beams, channels, samples, dtype, time_thresholds, n_time, policy, &ot, ct);
  if (st != RFIM_OK) return st;
  if (n_freq > 0) {
    st = validate(1, data, beams, channels, samples, dtype, freq_thresholds, n_freq, policy, &of, cf);
    if (st != RFIM_OK) return st;
  }
  if (!out) out = data;
  const size_t es = elem_size(dtype);
  const int64_t stride = ct.stride;
  const size_t beam_elems = (size_t)channels * (size_t)stride;
  const int per_chunk = host_chunk_beams(beams, channels, stride, es);
  const int nchunks = (beams + per_chunk - 1) / per_chunk;
  const int nslots = nchunks < kHostSlots ? nchunks : kHostSlots;
  const size_t slot_bytes = ((size_t)per_chunk * beam_elems * es + 255) & ~(size_t)255;
  HostStreams* hs = nullptr;
  if ((st = host_streams(hs)) != RFIM_OK) return st;
  void* dev[kHostSlots] = {nullptr, nullptr, nullptr};
  void* owned = nullptr;
  if (workspace) {
    if ((reinterpret_cast<uintptr_t>(workspace) & 255) != 0) return RFIM_ERR_INVALID;
    for (int i = 0; i < nslots; ++i) dev[i] = static_cast<char*>(workspace) + (size_t)i * slot_bytes;
  } else {
    CUDA_TRY(cudaMalloc(&owned, (size_t)nslots * slot_bytes));
    for (int i = 0; i < nslots; ++i) dev[i] = static_cast<char*>(owned) + (size_t)i * slot_bytes;
  }
  int rc = RFIM_OK;
  auto fail = [&](cudaError_t e, const char* what) { if (rc == RFIM_OK) rc = cuda_fail(e, what); };
  for (int ch = 0; ch < nchunks && rc == RFIM_OK; ++ch) {
    const int slot = ch % nslots;
    const int b0 = ch * per_chunk;
    const int nb = (beams - b0 < per_chunk) ? beams - b0 : per_chunk;
    const size_t rows = (size_t)nb * channels;
    const char* h_in = static_cast<const char*>(data) + (size_t)b0 * beam_elems * es;
    char* h_out = static_cast<char*>(out) + (size_t)b0 * beam_elems * es;
    cudaStream_t s = hs->s[slot];
    // dense rows: one linear copy (a 2-D copy of 12500-byte rows is markedly slower over PCIe)
    cudaError_t e = stride == samples
                        ? cudaMemcpyAsync(dev[slot], h_in, rows * (size_t)samples * es, cudaMemcpyHostToDevice, s)
                        : cudaMemcpy2DAsync(dev[slot], (size_t)stride * es, h_in, (size_t)stride * es,
                                            (size_t)samples * es, rows, cudaMemcpyHostToDevice, s);
    if (e != cudaSuccess) { fail(e, stride == samples ? "cudaMemcpyAsync(H2D)" : "cudaMemcpy2DAsync(H2D)"); break; }
    Call t = ct, f = cf;
    t.data = t.out = dev[slot]; t.beams = nb; t.stream = s; t.workspace = nullptr;
    if (n_freq > 0) { f.data = f.out = dev[slot]; f.beams = nb; f.stream = s; f.workspace = nullptr; }
    if (n_time > 0) {
      if ((st = run_time(t)) != RFIM_OK) { rc = st; break; }
    }
    if (n_freq > 0) {
      if ((st = run_freq(f)) != RFIM_OK) { rc = st; break; }
    }
    e = stride == samples
            ? cudaMemcpyAsync(h_out, dev[slot], rows * (size_t)samples * es, cudaMemcpyDeviceToHost, s)
            : cudaMemcpy2DAsync(h_out, (size_t)stride * es, dev[slot], (size_t)stride * es, (size_t)samples * es, rows,
                                cudaMemcpyDeviceToHost, s);
    if (e != cudaSuccess) { fail(e, stride == samples ? "cudaMemcpyAsync(D2H)" : "cudaMemcpy2DAsync(D2H)"); break; }
  }
  for (int i = 0; i < nslots; ++i) {
    cudaError_t e = cudaStreamSynchronize(hs->s[i]);
    if (e != cudaSuccess) fail(e, "cudaStreamSynchronize");
  }
  if (owned) cudaFree(owned);
  return rc;
}

size_t rfim_workspace_bytes(int op, int beams, int channels, int samples, rfim_dtype dtype,
                            int n_thresholds, rfim_replace policy, const rfim_opts* opts) {
  (void)n_thresholds; (void)policy;
  if (op == RFIM_OP_FREQ || op == RFIM_OP_TIME_FREQ) return 256;   // the FDSC tile dispenser (4 bytes used)
  if (op != RFIM_OP_HOST) return 0;                   // TDSC needs no scratch
  if (beams <= 0 || channels <= 0 || samples <= 0 || (dtype != RFIM_U8 && dtype != RFIM_F32)) return 0;
  const size_t es = elem_size(dtype);
  int64_t stride = (opts && opts->sample_stride) ? opts->sample_stride : samples;
  if (stride < samples) return 0;
  const int per_chunk = host_chunk_beams(beams, channels, stride, es);
  const int nchunks = (beams + per_chunk - 1) / per_chunk;
  const int nslots = nchunks < kHostSlots ? nchunks : kHostSlots;
  const size_t slot_bytes = ((size_t)per_chunk * (size_t)channels * (size_t)stride * es + 255) & ~(size_t)255;
  return (size_t)nslots * slot_bytes;
}


uint64_t rfim_launch_count(void) { return rfim_host::launches(); }
const char* rfim_last_variant(void) { return rfim_host::last_variant(); }
const char* rfim_last_cuda_error(void) { return rfim_host::last_cuda_error(); }
int rfim_version(void) { return RFIM_VERSION; }

const char* rfim_status_string(int status) {
  switch (status) {
    case RFIM_OK: return "ok";
    case RFIM_ERR_INVALID: return "invalid argument";
    case RFIM_ERR_UNSUPPORTED: return "unsupported: no kernel implements this request";
    case RFIM_ERR_CUDA: return "CUDA error (see rfim_last_cuda_error)";
    case RFIM_ERR_TOO_LARGE: return "too large: more tiles than the fixed scratch of the no-allocation entry point covers (RFIM_NOALLOC_MAX_TILES)";
    default: return "unknown status";
  }
}

}  // extern "C"

