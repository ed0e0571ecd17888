// rfim_noalloc.cu -- rfim_freq_sigma_cut_noalloc: the frequency-domain sigma cut (FDSC) for callers
// that cannot allocate device memory (code under CUDA graph capture, tight serving loops, harnesses that forbid
// cudaMalloc).
//
// The streaming FDSC kernel (fd_u8_quad.cuh) hands its tiles out through a ticket counter in device scratch memory.
// rfim_freq_sigma_cut takes that scratch from opts->workspace or, failing that, from the stream-ordered memory pool
// (cudaMallocAsync / cudaFreeAsync around the launch).  This entry point runs the same kernel with the scratch in a
// file-scope device array of fixed size: every GPU that loads the library holds these 256 bytes until the process
// exits, no call allocates or frees anything, and requests beyond the stated maximum are refused.
//
// All calls on a device share the array.  The ticket is cleared on the call's stream before every launch (the array
// keeps the last call's contents), so calls that follow one another on a stream are fine; calls that OVERLAP on the
// GPU (different streams, no dependency between them) race on the ticket and give wrong results.
#include "host.h"

#include <mutex>

namespace {

// the scratch: word 0 is the tile ticket of the launch in flight, the rest is reserved (rfim_workspace_bytes = 256)
static __device__ __align__(256) unsigned int g_noalloc_scratch[RFIM_NOALLOC_SCRATCH_BYTES / sizeof(unsigned int)];

constexpr int kMaxDevices = 64;

// In host code `g_noalloc_scratch` is a host-side stand-in, not a device address: the address a kernel may use is
// looked up once per device, with that device current.
int scratch_address(void** out) {
  static std::mutex mu;
  static void* addr[kMaxDevices] = {};
  int dev = 0;
  int st = rfim_host::current_device(dev);
  if (st != RFIM_OK) return st;
  if (dev < 0 || dev >= kMaxDevices) return RFIM_ERR_UNSUPPORTED;
  std::lock_guard<std::mutex> lock(mu);
  if (!addr[dev]) {
    void* p = nullptr;
    cudaError_t e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
    if (e != cudaSuccess) return rfim_host::cuda_fail(e, "cudaGetSymbolAddress(noalloc scratch)");
    if (!p || (reinterpret_cast<uintptr_t>(p) & 255) != 0) return RFIM_ERR_UNSUPPORTED;
    addr[dev] = p;
  }
  *out = addr[dev];
  return RFIM_OK;
}

}  // namespace

extern "C" int rfim_freq_sigma_cut_noalloc(void* data, int beams, int channels, int samples, rfim_dtype dtype,
                                           const double* thresholds, int n_thresholds, rfim_replace policy,
                                           const rfim_opts* opts) {
  // what the fixed scratch and its kernel cover; everything else is validated by rfim_freq_sigma_cut below
  if (!data || beams <= 0 || channels <= 0 || samples <= 0) return RFIM_ERR_INVALID;
  if (opts && (opts->workspace != nullptr || opts->variant != 0)) return RFIM_ERR_INVALID;   // the scratch is ours
  if (dtype != RFIM_U8 || policy != RFIM_REPLACE_MEAN) return RFIM_ERR_UNSUPPORTED;
  if (opts && opts->bin_size != 0 && opts->bin_size != channels) return RFIM_ERR_UNSUPPORTED;
  if (channels != 512 && channels != 1024 && channels != 1536 && channels != 2048) return RFIM_ERR_UNSUPPORTED;
  const int64_t tiles = (int64_t)beams * (((int64_t)samples + 127) / 128);
  if (tiles > (int64_t)RFIM_NOALLOC_MAX_TILES) return RFIM_ERR_TOO_LARGE;
  void* scratch = nullptr;
  int st = scratch_address(&scratch);
  if (st != RFIM_OK) return st;
  rfim_opts o;
  memset(&o, 0, sizeof(o));
  if (opts) o = *opts;
  o.workspace = scratch;                     // the tile dispenser: cleared on the stream by the launch
  o.variant = 17;                            // the streaming kernel or RFIM_ERR_UNSUPPORTED, never another path
  return rfim_freq_sigma_cut(data, beams, channels, samples, dtype, thresholds, n_thresholds, policy, &o);
}
