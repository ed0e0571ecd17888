// launch_fd_stream.cu -- geometry and launch of the streaming FDSC uint8 kernel (fd_u8_stream.cuh).
#include "host.h"
#include "fd_u8_stream.cuh"
#include "fd_u8_quad.cuh"
#include "fd_u8_qbin.cuh"

namespace rfim_host {

// ---- streaming kernel (fd_u8_stream.cuh): channel counts of 128 * {4, 8, 12, 16}, mean replacement, one bin or
// bins whose size is a multiple of 16 that divides the 32 * NCH channels one warp quartet owns
struct StreamPlan { int nch, slots, smem, nbins; bool binned, copy; };
bool plan_fd_u8_stream(const Call& c, StreamPlan& pl) {
  if (c.policy != RFIM_REPLACE_MEAN) return false;
  if (c.channels % 128 != 0) return false;
  pl.nch = c.channels / 128;
  if (pl.nch != 4 && pl.nch != 8 && pl.nch != 12 && pl.nch != 16) return false;
  const uintptr_t src = reinterpret_cast<uintptr_t>(c.data), dst = reinterpret_cast<uintptr_t>(c.out);
  if ((src & 3) != 0 || (dst & 3) != 0 || (c.stride & 3) != 0) return false;     // 32-bit word columns
  if ((int64_t)c.beams * c.channels / 4 > 0x7fffffff) return false;              // tensor coordinates
  if (!tensor_maps_available()) return false;
  pl.binned = c.bin_size != c.channels;
  pl.nbins = 0;
  if (pl.binned) {
    const int nb = c.bin_size;
    if (nb % 16 != 0 || nb > 256 || (32 * pl.nch) % nb != 0) return false;
    pl.nbins = c.channels / nb;
    if (pl.nbins > rfim::kFsMaxBins) return false;
  }
  if ((int64_t)c.beams * ((c.samples + rfim::kFsCols - 1) / rfim::kFsCols) >= 0x7fffffff) return false;   // tickets
  pl.copy = c.out != c.data;
  pl.slots = pl.binned ? 3 : 4;
  pl.smem = (int)rfim::fd_stream_smem_bytes(pl.slots, pl.nbins);
  return pl.smem <= kMaxSmem;
}

// The tile dispenser of a launch without caller workspace comes from the device's stream-ordered memory pool.  By
// default that pool hands all unused memory back to the OS at the next synchronisation, which turns the 256 bytes
// into an OS round trip per call: keep them (release threshold = maximum), once per device.
static int ticket_alloc(cudaStream_t stream, unsigned int** out) {
  static thread_local int prepared_dev = -1;
  int dev = 0;
  int st = current_device(dev);
  if (st != RFIM_OK) return st;
  if (prepared_dev != dev) {
    cudaMemPool_t pool;
    if (cudaDeviceGetDefaultMemPool(&pool, dev) == cudaSuccess) {
      unsigned long long keep = ~0ull;
      cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
    }
    prepared_dev = dev;
  }
  void* p = nullptr;
  CUDA_TRY(cudaMallocAsync(&p, 256, stream));
  *out = static_cast<unsigned int*>(p);
  return RFIM_OK;
}

using StreamKernel = void (*)(const rfim::FdStreamMaps, const rfim::FdStreamParams);

// one launch of a ticket-driven kernel: as many CTAs as are resident at once (at most one per tile), outputs
// cleared, the tile dispenser zeroed on the stream
template <typename Maps>
static int launch_ticketed(const Call& c, const char* name, void (*kernel)(const Maps, const rfim::FdStreamParams),
                           int threads, size_t smem, const Maps& maps, const rfim::FdStreamParams& P, int sms) {
  int st = ensure_smem(kernel, smem);
  if (st != RFIM_OK) return st;
  int occ = 0;
  if ((st = blocks_per_sm(kernel, threads, smem, occ)) != RFIM_OK) return st;
  if (occ < 1) return RFIM_ERR_UNSUPPORTED;
  int64_t grid = P.total_tiles;
  if (grid > (int64_t)sms * occ) grid = (int64_t)sms * occ;
  if ((st = clear_outputs(c)) != RFIM_OK) return st;
  // the tile dispenser: 4 bytes of zeroed device memory, the caller's (opts->workspace) or, failing that, taken from
  // and returned to the stream-ordered memory pool around the launch
  rfim::FdStreamParams Q = P;
  bool owned = false;
  if (c.workspace) {
    Q.ticket = static_cast<unsigned int*>(c.workspace);
  } else {
    if ((st = ticket_alloc(c.stream, &Q.ticket)) != RFIM_OK) return st;
    owned = true;
  }
  cudaError_t e = cudaMemsetAsync(Q.ticket, 0, sizeof(unsigned int), c.stream);
  if (e != cudaSuccess) {
    if (owned) cudaFreeAsync(Q.ticket, c.stream);
    return cuda_fail(e, "cudaMemsetAsync(ticket)");
  }
  st = launch(name, kernel, dim3((unsigned)grid), dim3((unsigned)threads), smem, c.stream, 0, maps, Q);
  if (owned) {
    e = cudaFreeAsync(Q.ticket, c.stream);
    if (e != cudaSuccess && st == RFIM_OK) st = cuda_fail(e, "cudaFreeAsync(ticket)");
  }
  return st;
}

// parameters and tensor maps every ticket-driven kernel shares (boxes of 8 class rows x 144 bytes)
static bool stream_params(const Call& c, rfim::FdStreamParams& P, rfim::FdStreamMaps& maps) {
  memset(&P, 0, sizeof(P));
  P.src = static_cast<const uint8_t*>(c.data);
  P.dst = static_cast<uint8_t*>(c.out);
  P.stride = c.stride;
  P.beams = c.beams; P.C = c.channels; P.S = c.samples;
  P.beam0 = 0;
  P.n_thr = c.n_thr;
  for (int i = 0; i < c.n_thr; ++i) P.p[i] = quantise(c.thr[i]);
  P.flags = c.flags;
  P.counts = c.counts;
  P.tiles_per_beam = (c.samples + rfim::kFsCols - 1) / rfim::kFsCols;
  P.total_tiles = (int64_t)P.tiles_per_beam * c.beams;
  P.invC = (uint32_t)((((uint64_t)1 << 32) + (uint64_t)c.channels - 1) / (uint64_t)c.channels);
  P.nb = c.bin_size;
  P.nbins = c.channels / c.bin_size;
  P.inv_nb = (uint32_t)((((uint64_t)1 << 32) + (uint64_t)P.nb - 1) / (uint64_t)P.nb);
  P.inv_2nb = (uint32_t)((((uint64_t)1 << 32) + 2 * (uint64_t)P.nb - 1) / (2 * (uint64_t)P.nb));
  ClassMaps cm;
  // No L2 promotion: a box row is the 144-byte superset of 128 columns; promoted to whole 128-byte lines it costs
  // two lines (256 bytes) of DRAM traffic, because the half-used line is rarely still in L2 when the neighbouring
  // tile asks for it (measured: 18.2 GB read for a 9.2 GB batch with 128-byte promotion).
  if (!encode_class_maps(P.src, c.stride, c.samples, (int64_t)c.beams * c.channels, rfim::kFsPitchW * 4,
                         rfim::kFsBoxRows, CU_TENSOR_MAP_L2_PROMOTION_NONE, cm))
    return false;
  for (int k = 0; k < 4; ++k) { maps.src[k] = cm.m[k]; P.off[k] = cm.off[k]; }
  return true;
}

template <int NCH>
int launch_fd_stream_n(const Call& c, const StreamPlan& pl, const rfim::FdStreamMaps& maps,
                       const rfim::FdStreamParams& P, int sms) {
  StreamKernel kernel;
  const char* name;
  if (pl.binned) {
    kernel = pl.copy ? rfim::fd_u8_stream_kernel<NCH, 3, true, true> : rfim::fd_u8_stream_kernel<NCH, 3, true, false>;
    name = pl.copy ? "fd_u8_stream_binned_copy" : "fd_u8_stream_binned";
  } else {
    kernel = pl.copy ? rfim::fd_u8_stream_kernel<NCH, 4, false, true> : rfim::fd_u8_stream_kernel<NCH, 4, false, false>;
    name = pl.copy ? "fd_u8_stream_copy" : "fd_u8_stream";
  }
  return launch_ticketed(c, name, kernel, rfim::kFsThreads, (size_t)pl.smem, maps, P, sms);
}

int launch_fd_stream(const Call& c, const StreamPlan& pl, int sms) {
  rfim::FdStreamParams P;
  rfim::FdStreamMaps maps;
  if (!stream_params(c, P, maps)) return RFIM_ERR_UNSUPPORTED;
  P.nbins = pl.nbins;
  switch (pl.nch) {
    case 4: return launch_fd_stream_n<4>(c, pl, maps, P, sms);
    case 8: return launch_fd_stream_n<8>(c, pl, maps, P, sms);
    case 12: return launch_fd_stream_n<12>(c, pl, maps, P, sms);
    default: return launch_fd_stream_n<16>(c, pl, maps, P, sms);
  }
}

// ---- one warp per alignment class (fd_u8_quad.cuh): one bin, channel counts of 128 * {4, 8, 12, 16}
template <int NBQ>
int launch_fd_quad_n(const Call& c, bool copy, const rfim::FdStreamMaps& maps, const rfim::FdStreamParams& P, int sms) {
  // a ring of 4 boxes per warp and four CTAs per SM (measured on config 4: 3.63 ms; a ring of 3 with five CTAs per
  // SM 3.76 ms, a ring of 5 3.79 ms)
  constexpr int ring = 4;
  StreamKernel kernel = copy ? rfim::fd_u8_quad_kernel<NBQ, true, ring> : rfim::fd_u8_quad_kernel<NBQ, false, ring>;
  return launch_ticketed(c, copy ? "fd_u8_quad_copy" : "fd_u8_quad", kernel, rfim::kFqThreads,
                         rfim::fd_quad_smem_bytes(NBQ, ring), maps, P, sms);
}

int try_fd_u8_quad(const Call& c, int sms) {
  StreamPlan pl;
  if (!plan_fd_u8_stream(c, pl) || pl.binned) return RFIM_ERR_UNSUPPORTED;   // same geometry limits, one bin only
  rfim::FdStreamParams P;
  rfim::FdStreamMaps maps;
  if (!stream_params(c, P, maps)) return RFIM_ERR_UNSUPPORTED;
  switch (pl.nch) {                                    // channels / 128
    case 4: return launch_fd_quad_n<4>(c, pl.copy, maps, P, sms);
    case 8: return launch_fd_quad_n<8>(c, pl.copy, maps, P, sms);
    case 12: return launch_fd_quad_n<12>(c, pl.copy, maps, P, sms);
    default: return launch_fd_quad_n<16>(c, pl.copy, maps, P, sms);
  }
}

// ---- one streaming pass per step with per-bin sums (fd_u8_qbin.cuh): channel counts of 256 * {2, 4, 6, 8}, bins of
// a multiple of 16 channels (at most 256) that divide half the channels
using QbinKernel = void (*)(const rfim::FdQbMaps, const rfim::FdStreamParams);

template <int NB>
int launch_fd_qbin_n(const Call& c, bool copy, const rfim::FdQbMaps& maps, const rfim::FdStreamParams& P, int sms) {
  const bool outputs = c.flags != nullptr || c.counts != nullptr;
  QbinKernel kernel = copy ? (outputs ? rfim::fd_u8_qbin_kernel<NB, true, true> : rfim::fd_u8_qbin_kernel<NB, true, false>)
                           : (outputs ? rfim::fd_u8_qbin_kernel<NB, false, true> : rfim::fd_u8_qbin_kernel<NB, false, false>);
  size_t smem = rfim::fd_qbin_smem_bytes(P.nbins);
  if (smem > (size_t)kMaxSmem) return RFIM_ERR_UNSUPPORTED;
  // Three CTAs per SM are faster per SM than two (96 beams, bins of 32: 1.70 vs 1.88 ms), but a tile then takes a CTA
  // a third longer (80 vs 59 us), and a short batch is a handful of tile times: 12 beams are 1176 tiles = 4 full
  // rounds of 2 x 148 CTAs (0.262 ms) or 2.65 rounds of 3 x 148 (0.290 ms).  Two per SM (asked for through the
  // shared-memory size) whenever its whole rounds are not more than 4 / 3 of the other's.
  const size_t two_per_sm = (size_t)(kMaxSmem + 1024) / 3;          // more than a third of an SM's shared memory
  if (smem < two_per_sm) {
    const int64_t w2 = (P.total_tiles + 2 * sms - 1) / (2 * sms), w3 = (P.total_tiles + 3 * sms - 1) / (3 * sms);
    if (3 * w2 <= 4 * w3) smem = two_per_sm;
  }
  return launch_ticketed(c, copy ? "fd_u8_qbin_copy" : "fd_u8_qbin", kernel, rfim::kQbThreads, smem, maps, P, sms);
}

int try_fd_u8_qbin(const Call& c, int sms) {
  if (c.policy != RFIM_REPLACE_MEAN || c.bin_size == c.channels || c.n_thr < 1) return RFIM_ERR_UNSUPPORTED;
  const int nb = c.bin_size;
  if (c.channels % 256 != 0 || nb % 16 != 0 || nb > 256 || (c.channels / 2) % nb != 0) return RFIM_ERR_UNSUPPORTED;
  const uintptr_t src = reinterpret_cast<uintptr_t>(c.data), dst = reinterpret_cast<uintptr_t>(c.out);
  if ((src & 3) != 0 || (dst & 3) != 0 || (c.stride & 3) != 0) return RFIM_ERR_UNSUPPORTED;   // 32-bit word columns
  if ((int64_t)c.beams * c.channels / 4 > 0x7fffffff) return RFIM_ERR_UNSUPPORTED;            // tensor coordinates
  if ((int64_t)c.beams * ((c.samples + rfim::kFsCols - 1) / rfim::kFsCols) >= 0x7fffffff) return RFIM_ERR_UNSUPPORTED;
  if (!tensor_maps_available()) return RFIM_ERR_UNSUPPORTED;
  const bool copy = c.out != c.data;
  rfim::FdStreamParams P;
  rfim::FdStreamMaps smaps;
  if (!stream_params(c, P, smaps)) return RFIM_ERR_UNSUPPORTED;
  rfim::FdQbMaps maps;
  for (int k = 0; k < 4; ++k) { maps.src[k] = smaps.src[k]; maps.dst[k] = smaps.src[k]; P.off_dst[k] = P.off[k]; }
  if (copy) {                                          // the iteration passes stream the destination
    ClassMaps cm;
    if (!encode_class_maps(P.dst, c.stride, c.samples, (int64_t)c.beams * c.channels, rfim::kFsPitchW * 4,
                           rfim::kFsBoxRows, CU_TENSOR_MAP_L2_PROMOTION_NONE, cm))
      return RFIM_ERR_UNSUPPORTED;
    for (int k = 0; k < 4; ++k) { maps.dst[k] = cm.m[k]; P.off_dst[k] = cm.off[k]; }
  }
  switch (c.channels / 256) {
    case 2: return launch_fd_qbin_n<8>(c, copy, maps, P, sms);
    case 4: return launch_fd_qbin_n<16>(c, copy, maps, P, sms);
    case 6: return launch_fd_qbin_n<24>(c, copy, maps, P, sms);
    case 8: return launch_fd_qbin_n<32>(c, copy, maps, P, sms);
    default: return RFIM_ERR_UNSUPPORTED;
  }
}

int try_fd_u8_stream(const Call& c, int sms) {
  StreamPlan sp;
  if (!plan_fd_u8_stream(c, sp)) return RFIM_ERR_UNSUPPORTED;
  return launch_fd_stream(c, sp, sms);
}

}  // namespace rfim_host
