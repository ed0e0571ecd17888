// rfim_api.cu -- the C ABI of librfim (include/rfim.h): argument checks, variant selection,
// launches.  No CPU fallback: every step of the path runs in the kernels of this directory.
#include "../../include/rfim.h"

#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstring>

#include "common.cuh"
#include "fd_u8.cuh"
#include "td_f32.cuh"
#include "td_u8.cuh"

namespace {

std::atomic<uint64_t> g_launches{0};
thread_local char t_cuda_error[256] = "";
thread_local const char* t_variant = "";

constexpr int kMaxSmem = 227 * 1024;   // opt-in dynamic shared memory per CTA on sm_100

int cuda_fail(cudaError_t e, const char* what) {
  snprintf(t_cuda_error, sizeof(t_cuda_error), "%s: %s", what, cudaGetErrorString(e));
  return RFIM_ERR_CUDA;
}
#define CUDA_TRY(expr)                                   \
  do {                                                   \
    cudaError_t e_ = (expr);                             \
    if (e_ != cudaSuccess) return cuda_fail(e_, #expr);  \
  } while (0)

struct DevInfo { int sms = 0; };
int dev_info(DevInfo& d) {
  int dev = 0;
  CUDA_TRY(cudaGetDevice(&dev));
  CUDA_TRY(cudaDeviceGetAttribute(&d.sms, cudaDevAttrMultiProcessorCount, dev));
  return RFIM_OK;
}

size_t elem_size(rfim_dtype t) { return t == RFIM_U8 ? 1 : 4; }

// p = round-half-even(k * 2^16): k * 65536 is exact, nearbyint rounds half to even (default mode)
uint32_t quantise(double k) { return (uint32_t)std::nearbyint(k * 65536.0); }

struct Call {
  void* data; void* out;
  int beams, channels, samples;
  rfim_dtype dtype;
  const double* thr; int n_thr;
  rfim_replace policy;
  int64_t stride; int window; int bin_size;
  uint8_t* flags; unsigned long long* counts;
  cudaStream_t stream; void* workspace; int variant; int reserved_team;
};

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
  if (z.variant < 0 || z.variant > 4) return RFIM_ERR_INVALID;
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
  c.variant = z.variant;
  c.reserved_team = 0;
  if (z.variant == 3 || z.variant == 4) { c.reserved_team = z.variant - 2; c.variant = 2; }
  return RFIM_OK;
}

// flags / counts are defined as "overwritten": clear them on the stream before the kernel adds to them
int clear_outputs(const Call& c) {
  if (c.flags)
    CUDA_TRY(cudaMemsetAsync(c.flags, 0, (size_t)c.beams * c.channels * c.samples, c.stream));
  if (c.counts && c.n_thr > 0)
    CUDA_TRY(cudaMemsetAsync(c.counts, 0, sizeof(unsigned long long) * c.n_thr, c.stream));
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

int after_launch(const char* name) {
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return cuda_fail(e, name);
  g_launches.fetch_add(1, std::memory_order_relaxed);
  t_variant = name;
  return RFIM_OK;
}

// ------------------------------------------------------------------------------------------ TD u8
struct StagedPlan { int nteams, team, slot_bytes, queue_entries, smem; };

bool plan_td_u8_staged(const Call& c, StagedPlan& pl) {
  if (c.window != c.samples || c.policy != RFIM_REPLACE_MEAN) return false;
  // every row must have the same misalignment in src and dst for the aligned interior to match
  if (((reinterpret_cast<uintptr_t>(c.data) ^ reinterpret_cast<uintptr_t>(c.out)) & 15) != 0) return false;
  if (c.samples > 65000) return false;                    // 32-bit S, Q totals inside the kernel
  pl.slot_bytes = (c.samples + 30 + 15) & ~15;
  pl.queue_entries = ((pl.slot_bytes / 16) + 3) & ~3;
  // per team: one slot, one hit queue, one control block; sixteen teams keep sixteen rows in flight
  const int per_team = pl.slot_bytes + pl.queue_entries * 2 + rfim::kCtrlBytes;
  pl.nteams = kMaxSmem / per_team;
  if (pl.nteams > 16) pl.nteams = 16;
  if (pl.nteams < 4) return false;
  pl.smem = pl.nteams * per_team;
  pl.team = 1;                                            // warps per row (TD kernel: measured)
  if (c.variant == 2 && c.reserved_team > 0) pl.team = c.reserved_team;
  return true;
}

int launch_td_u8(const Call& c) {
  rfim::TdU8Params P;
  memset(&P, 0, sizeof(P));
  P.src = static_cast<const uint8_t*>(c.data);
  P.dst = static_cast<uint8_t*>(c.out);
  P.rows = (int64_t)c.beams * c.channels;
  P.stride = c.stride;
  P.S = c.samples;
  P.window = c.window;
  P.n_thr = c.n_thr;
  P.policy = (int)c.policy;
  for (int i = 0; i < c.n_thr; ++i) { P.p[i] = quantise(c.thr[i]); P.pf[i] = (float)P.p[i] * (1.0f / 65536.0f); }
  P.flags = c.flags;
  P.counts = c.counts;
  DevInfo dv;
  int st = dev_info(dv);
  if (st != RFIM_OK) return st;

  StagedPlan pl;
  const bool can_stage = plan_td_u8_staged(c, pl);
  if (c.variant == 2 && !can_stage) return RFIM_ERR_UNSUPPORTED;
  if (can_stage && c.variant != 1) {
    P.slot_bytes = pl.slot_bytes;
    P.queue_entries = pl.queue_entries;
    void (*kernel)(const rfim::TdU8Params);
    if (pl.team == 2) kernel = c.flags ? rfim::td_u8_staged_kernel<2, true> : rfim::td_u8_staged_kernel<2, false>;
    else kernel = c.flags ? rfim::td_u8_staged_kernel<1, true> : rfim::td_u8_staged_kernel<1, false>;
    const int threads = pl.nteams * pl.team * 32;
    CUDA_TRY(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, pl.smem));
    int occ = 0;
    CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kernel, threads, pl.smem));
    if (occ < 1) occ = 1;
    int64_t grid = (P.rows + pl.nteams - 1) / pl.nteams;
    if (grid > (int64_t)dv.sms * occ) grid = (int64_t)dv.sms * occ;
    if ((st = clear_outputs(c)) != RFIM_OK) return st;
    kernel<<<(unsigned)grid, threads, pl.smem, c.stream>>>(P);
    return after_launch(pl.team == 2 ? "td_u8_staged_team2" : "td_u8_staged");
  }
  int64_t grid = P.rows;
  if (grid > (int64_t)dv.sms * 32) grid = (int64_t)dv.sms * 32;
  if ((st = clear_outputs(c)) != RFIM_OK) return st;
  rfim::td_u8_generic_kernel<<<(unsigned)grid, rfim::kGenericThreads, 0, c.stream>>>(P);
  return after_launch("td_u8_generic");
}

// ------------------------------------------------------------------------------------------ FD u8
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_tiled_fn() {
  static EncodeTiledFn fn = [] {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess ||
        q != cudaDriverEntryPointSuccess)
      p = nullptr;
    return reinterpret_cast<EncodeTiledFn>(p);
  }();
  return fn;
}

struct FdPlan { int ts, m, rows_per_class, box_rows, smem; bool exact; };

template <int Ts, bool kExact>
size_t fd_smem_bytes(int C) {
  const size_t row_bytes = kExact ? Ts : Ts + 16;
  return (((size_t)C * row_bytes + 127) & ~(size_t)127) + sizeof(rfim::FdSmem<Ts>);
}
size_t fd_smem_for(int ts, int C) {
  switch (ts) {
    case 128: return fd_smem_bytes<128, true>(C);
    case 64: return fd_smem_bytes<64, true>(C);
    case 32: return fd_smem_bytes<32, true>(C);
    case 112: return fd_smem_bytes<112, false>(C);
    default: return fd_smem_bytes<48, false>(C);
  }
}

// Tile geometry for the request, or false when only the generic kernel can run it.  `big` prefers the
// widest tile that fits one CTA per SM over a narrower one with two CTAs per SM (variant 3).
bool plan_fd_u8_tile(const Call& c, bool big, FdPlan& pl) {
  if (c.policy != RFIM_REPLACE_MEAN || c.bin_size != c.channels) return false;
  int m = 1;
  while ((((int64_t)m * c.stride) & 15) != 0) m <<= 1;       // rows per 16-byte alignment period
  if (m > rfim::kFdMaxClasses || c.channels % m != 0) return false;
  if (c.channels > 60000) return false;                      // 32-bit column totals inside the kernel
  const uintptr_t src = reinterpret_cast<uintptr_t>(c.data), dst = reinterpret_cast<uintptr_t>(c.out);
  pl.exact = (m == 1) && ((src | dst) & 15) == 0;
  if (!pl.exact && ((src | dst) & 3) != 0) return false;     // 32-bit stores of the tile
  pl.m = m;
  pl.rows_per_class = c.channels / m;
  static const int exact_ts[3] = {128, 64, 32}, over_ts[2] = {112, 48};
  const int* cand = pl.exact ? exact_ts : over_ts;
  const int ncand = pl.exact ? 3 : 2;
  const size_t half = (size_t)(kMaxSmem + 1024) / 2 - 1024;  // two CTAs per SM (1 KB reserved per CTA)
  // TMA boxes: rows per box divides the class, <= 256, and every box lands 128-byte aligned in shared memory
  auto boxes_for = [&](int ts) {
    const int row_bytes = pl.exact ? ts : ts + 16;
    if (m > 1 && ((int64_t)pl.rows_per_class * row_bytes) % 128 != 0) return 0;
    int best = 0;
    for (int d = 1; d <= 256 && d <= pl.rows_per_class; ++d)
      if (pl.rows_per_class % d == 0 && (d * row_bytes) % 128 == 0) best = d;
    if (pl.rows_per_class == best) return best;                // a single box needs no alignment of its size
    if (best == 0 && pl.rows_per_class <= 256) return pl.rows_per_class;
    return (best && pl.rows_per_class / best <= 64) ? best : 0;
  };
  pl.ts = 0;
  for (int pass = big ? 1 : 0; pass < 2 && !pl.ts; ++pass)
    for (int i = 0; i < ncand && !pl.ts; ++i)
      if (fd_smem_for(cand[i], c.channels) <= (pass == 0 ? half : (size_t)kMaxSmem) && boxes_for(cand[i]) > 0)
        pl.ts = cand[i];
  if (!pl.ts) return false;
  pl.box_rows = boxes_for(pl.ts);
  pl.smem = (int)fd_smem_for(pl.ts, c.channels);
  return true;
}

// one 2-D tensor per alignment class r: rows r, r+m, r+2m, ... of the [beams*channels][pitch] matrix,
// origin rounded down to 16 bytes (off[r] bytes before the row start)
bool encode_fd_maps(const Call& c, const FdPlan& pl, uint8_t* base, CUtensorMap* maps, int* off) {
  EncodeTiledFn enc = encode_tiled_fn();
  if (!enc) return false;
  for (int r = 0; r < pl.m; ++r) {
    const uintptr_t addr = reinterpret_cast<uintptr_t>(base) + (uintptr_t)r * (uintptr_t)c.stride;
    off[r] = (int)(addr & 15);
    cuuint64_t dims[2] = {(cuuint64_t)c.samples + (cuuint64_t)off[r],
                          (cuuint64_t)c.beams * (cuuint64_t)pl.rows_per_class};
    cuuint64_t strides[1] = {(cuuint64_t)pl.m * (cuuint64_t)c.stride};
    cuuint32_t box[2] = {(cuuint32_t)(pl.exact ? pl.ts : pl.ts + 16), (cuuint32_t)pl.box_rows};
    cuuint32_t estr[2] = {1, 1};
    if (enc(&maps[r], CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, reinterpret_cast<void*>(addr - off[r]), dims, strides, box,
            estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
      return false;
  }
  return true;
}

template <int Ts, bool kExact>
int launch_fd_tile(const Call& c, const FdPlan& pl, const rfim::FdMaps& maps, rfim::FdU8Params& P, int sms,
                   const char* name) {
  auto kernel = rfim::fd_u8_tile_kernel<Ts, kExact>;
  CUDA_TRY(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, pl.smem));
  int occ = 0;
  CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kernel, 4 * Ts, pl.smem));
  if (occ < 1) occ = 1;
  int64_t grid = P.total_tiles;
  if (grid > (int64_t)sms * occ) grid = (int64_t)sms * occ;
  int st = clear_outputs(c);
  if (st != RFIM_OK) return st;
  kernel<<<(unsigned)grid, 4 * Ts, pl.smem, c.stream>>>(maps, P);
  return after_launch(name);
}

int launch_fd_u8(const Call& c) {
  rfim::FdU8Params P;
  memset(&P, 0, sizeof(P));
  P.src = static_cast<const uint8_t*>(c.data);
  P.dst = static_cast<uint8_t*>(c.out);
  P.stride = c.stride;
  P.beams = c.beams; P.C = c.channels; P.S = c.samples;
  P.n_thr = c.n_thr;
  for (int i = 0; i < c.n_thr; ++i) { P.p[i] = quantise(c.thr[i]); P.pf[i] = (float)P.p[i] * (1.0f / 65536.0f); }
  P.flags = c.flags;
  P.counts = c.counts;
  DevInfo dv;
  int st = dev_info(dv);
  if (st != RFIM_OK) return st;

  FdPlan pl;
  bool can_tile = c.variant != 1 && plan_fd_u8_tile(c, c.reserved_team == 1, pl);
  rfim::FdMaps maps;
  if (can_tile) {
    int off_dst[rfim::kFdMaxClasses] = {0, 0, 0, 0};
    can_tile = encode_fd_maps(c, pl, static_cast<uint8_t*>(c.data), maps.src, P.off) &&
               (!pl.exact || encode_fd_maps(c, pl, static_cast<uint8_t*>(c.out), maps.dst, off_dst));
  }
  if (c.variant == 2 && !can_tile) return RFIM_ERR_UNSUPPORTED;
  if (can_tile) {
    P.m = pl.m; P.rows_per_class = pl.rows_per_class; P.box_rows = pl.box_rows;
    P.tiles_per_beam = (c.samples + pl.ts - 1) / pl.ts;
    P.total_tiles = (int64_t)P.tiles_per_beam * c.beams;
    switch (pl.ts) {
      case 128: return launch_fd_tile<128, true>(c, pl, maps, P, dv.sms, "fd_u8_tile128");
      case 64: return launch_fd_tile<64, true>(c, pl, maps, P, dv.sms, "fd_u8_tile64");
      case 32: return launch_fd_tile<32, true>(c, pl, maps, P, dv.sms, "fd_u8_tile32");
      case 112: return launch_fd_tile<112, false>(c, pl, maps, P, dv.sms, "fd_u8_tile112x");
      default: return launch_fd_tile<48, false>(c, pl, maps, P, dv.sms, "fd_u8_tile48x");
    }
  }
  if (c.policy != RFIM_REPLACE_MEAN || c.bin_size != c.channels) return RFIM_ERR_UNSUPPORTED;
  const int64_t ncol = (int64_t)c.beams * c.samples;
  int64_t grid = (ncol + rfim::kFdGenericThreads - 1) / rfim::kFdGenericThreads;
  if (grid > (int64_t)dv.sms * 16) grid = (int64_t)dv.sms * 16;
  if ((st = clear_outputs(c)) != RFIM_OK) return st;
  rfim::fd_u8_generic_kernel<<<(unsigned)grid, rfim::kFdGenericThreads, 0, c.stream>>>(P);
  return after_launch("fd_u8_generic");
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
  if (c.n_thr == 0) {
    if ((st = clear_outputs(c)) != RFIM_OK) return st;
    return copy_through(c);
  }
  if (dtype == RFIM_U8) return launch_td_u8(c);
  return RFIM_ERR_UNSUPPORTED;
}

int rfim_freq_sigma_cut(void* data, int beams, int channels, int samples, rfim_dtype dtype,
                        const double* thresholds, int n_thresholds, rfim_replace policy,
                        const rfim_opts* opts) {
  Call c;
  int st = validate(1, data, beams, channels, samples, dtype, thresholds, n_thresholds, policy, opts, c);
  if (st != RFIM_OK) return st;
  if (c.n_thr == 0) {
    if ((st = clear_outputs(c)) != RFIM_OK) return st;
    return copy_through(c);
  }
  if (dtype == RFIM_U8) return launch_fd_u8(c);
  return RFIM_ERR_UNSUPPORTED;
}

int rfim_sigma_cut_host(void* data, void* out, int beams, int channels, int samples, rfim_dtype dtype,
                        const double* time_thresholds, int n_time,
                        const double* freq_thresholds, int n_freq,
                        rfim_replace policy, const rfim_opts* opts) {
  // validate exactly as the device entry points do (the host pointers are never dereferenced here)
  Call ct, cf;
  int st = validate(0, data, beams, channels, samples, dtype, time_thresholds, n_time, policy, opts, ct);
  if (st != RFIM_OK) return st;
  st = validate(1, data, beams, channels, samples, dtype, freq_thresholds, n_freq, policy, opts, cf);
  if (st != RFIM_OK) return st;
  if (opts && (opts->out || opts->flags || opts->counts || opts->stream || opts->workspace)) return RFIM_ERR_INVALID;
  if (!out) out = data;
  const size_t es = elem_size(dtype);
  const int64_t stride = ct.stride;
  const size_t beam_elems = (size_t)channels * (size_t)stride;
  // chunk of whole beams, about 128 MiB: long enough copies for full PCIe rate, short enough to overlap
  int per_chunk = (int)((size_t)(128u << 20) / (beam_elems * es));
  if (per_chunk < 1) per_chunk = 1;
  if (per_chunk > beams) per_chunk = beams;
  const int nchunks = (beams + per_chunk - 1) / per_chunk;
  constexpr int kSlots = 3;
  const int nslots = nchunks < kSlots ? nchunks : kSlots;
  void* dev[kSlots] = {nullptr, nullptr, nullptr};
  cudaStream_t streams[kSlots] = {nullptr, nullptr, nullptr};
  int rc = RFIM_OK;
  auto fail = [&](cudaError_t e, const char* what) { if (rc == RFIM_OK) rc = cuda_fail(e, what); };
  for (int i = 0; i < nslots && rc == RFIM_OK; ++i) {
    cudaError_t e = cudaMalloc(&dev[i], (size_t)per_chunk * beam_elems * es);
    if (e != cudaSuccess) { fail(e, "cudaMalloc(staging)"); break; }
    e = cudaStreamCreateWithFlags(&streams[i], cudaStreamNonBlocking);
    if (e != cudaSuccess) fail(e, "cudaStreamCreate");
  }
  rfim_opts o;
  memset(&o, 0, sizeof(o));
  if (opts) { o.sample_stride = opts->sample_stride; o.window = opts->window; o.bin_size = opts->bin_size; }
  for (int ch = 0; ch < nchunks && rc == RFIM_OK; ++ch) {
    const int slot = ch % nslots;
    const int b0 = ch * per_chunk;
    const int nb = (beams - b0 < per_chunk) ? beams - b0 : per_chunk;
    const size_t rows = (size_t)nb * channels;
    const char* h_in = static_cast<const char*>(data) + (size_t)b0 * beam_elems * es;
    char* h_out = static_cast<char*>(out) + (size_t)b0 * beam_elems * es;
    cudaError_t e = cudaMemcpy2DAsync(dev[slot], (size_t)stride * es, h_in, (size_t)stride * es, (size_t)samples * es,
                                      rows, cudaMemcpyHostToDevice, streams[slot]);
    if (e != cudaSuccess) { fail(e, "cudaMemcpy2DAsync(H2D)"); break; }
    o.stream = streams[slot];
    if (n_time > 0) {
      st = rfim_time_sigma_cut(dev[slot], nb, channels, samples, dtype, time_thresholds, n_time, policy, &o);
      if (st != RFIM_OK) { rc = st; break; }
    }
    if (n_freq > 0) {
      st = rfim_freq_sigma_cut(dev[slot], nb, channels, samples, dtype, freq_thresholds, n_freq, policy, &o);
      if (st != RFIM_OK) { rc = st; break; }
    }
    e = cudaMemcpy2DAsync(h_out, (size_t)stride * es, dev[slot], (size_t)stride * es, (size_t)samples * es, rows,
                          cudaMemcpyDeviceToHost, streams[slot]);
    if (e != cudaSuccess) { fail(e, "cudaMemcpy2DAsync(D2H)"); break; }
  }
  for (int i = 0; i < nslots; ++i) {
    if (streams[i]) {
      cudaError_t e = cudaStreamSynchronize(streams[i]);
      if (e != cudaSuccess) fail(e, "cudaStreamSynchronize");
      cudaStreamDestroy(streams[i]);
    }
    if (dev[i]) cudaFree(dev[i]);
  }
  return rc;
}

size_t rfim_workspace_bytes(int op, int beams, int channels, int samples, rfim_dtype dtype,
                            int n_thresholds, rfim_replace policy, const rfim_opts* opts) {
  (void)op; (void)beams; (void)channels; (void)samples; (void)dtype; (void)n_thresholds; (void)policy; (void)opts;
  return 0;
}

uint64_t rfim_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }
const char* rfim_last_variant(void) { return t_variant; }
const char* rfim_last_cuda_error(void) { return t_cuda_error; }
int rfim_version(void) { return RFIM_VERSION; }

const char* rfim_status_string(int status) {
  switch (status) {
    case RFIM_OK: return "ok";
    case RFIM_ERR_INVALID: return "invalid argument";
    case RFIM_ERR_UNSUPPORTED: return "unsupported: no kernel implements this request";
    case RFIM_ERR_CUDA: return "CUDA error (see rfim_last_cuda_error)";
    default: return "unknown status";
  }
}

}  // extern "C"
