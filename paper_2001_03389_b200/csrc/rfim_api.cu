// rfim_api.cu -- the C ABI of librfim (include/rfim.h): argument checks, variant selection,
// launches.  No CPU fallback: every step of the path runs in the kernels of this directory.
#include "../../include/rfim.h"

#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <map>
#include <mutex>
#include <tuple>

#include "common.cuh"
#include "fd_u8.cuh"
#include "fd_f32.cuh"
#include "fd_u8_binned.cuh"
#include "fd_u8_stream.cuh"
#include "fd_u8_strip.cuh"
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

// ------------------------------------------------------------------------------ per-process caches
// Launch attributes do not depend on the data: shared-memory opt-in and occupancy are set / queried once per
// (device, kernel, block size, shared memory) and remembered, so a small real-time call (12 beams, ~0.1 ms)
// pays for the launch only.
std::mutex g_cache_mutex;
std::map<std::tuple<int, const void*>, int> g_smem_set;                       // largest opt-in so far
std::map<std::tuple<int, const void*, int, size_t, int>, int> g_occupancy;    // blocks (or clusters) per device
std::map<int, int> g_sms;

int current_device(int& dev) {
  CUDA_TRY(cudaGetDevice(&dev));
  return RFIM_OK;
}
int sm_count(int& sms) {
  int dev = 0;
  int st = current_device(dev);
  if (st != RFIM_OK) return st;
  std::lock_guard<std::mutex> lock(g_cache_mutex);
  auto it = g_sms.find(dev);
  if (it == g_sms.end()) {
    int n = 0;
    CUDA_TRY(cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev));
    it = g_sms.emplace(dev, n).first;
  }
  sms = it->second;
  return RFIM_OK;
}
template <typename K>
int ensure_smem(K kernel, size_t bytes) {
  int dev = 0;
  int st = current_device(dev);
  if (st != RFIM_OK) return st;
  std::lock_guard<std::mutex> lock(g_cache_mutex);
  int& have = g_smem_set[std::make_tuple(dev, reinterpret_cast<const void*>(kernel))];
  if ((int)bytes > have) {
    CUDA_TRY(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
    have = (int)bytes;
  }
  return RFIM_OK;
}
// resident CTAs per SM of a plain (non-cluster) kernel
template <typename K>
int blocks_per_sm(K kernel, int threads, size_t smem, int& occ) {
  int dev = 0;
  int st = current_device(dev);
  if (st != RFIM_OK) return st;
  std::lock_guard<std::mutex> lock(g_cache_mutex);
  const auto key = std::make_tuple(dev, reinterpret_cast<const void*>(kernel), threads, smem, 0);
  auto it = g_occupancy.find(key);
  if (it == g_occupancy.end()) {
    int n = 0;
    CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, kernel, threads, smem));
    it = g_occupancy.emplace(key, n).first;
  }
  occ = it->second;
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
  bool keep_outputs;                       // chain: flags / counts were prepared by the caller, do not clear them
};

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
  if (z.variant < 0 || z.variant > 16 || (z.variant >= 5 && z.variant <= 12)) return RFIM_ERR_INVALID;
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

// flags / counts are defined as "overwritten": clear them on the stream before the kernel adds to them
int clear_outputs(const Call& c) {
  if (c.keep_outputs) return RFIM_OK;
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

// One launch.  cudaLaunchKernelEx reports the error of THIS launch: an error some earlier, unrelated work left
// pending in the runtime is neither consumed nor blamed on this call.
template <typename... KArgs, typename... Args>
int launch(const char* name, void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t stream,
           int cluster, Args&&... args) {
  cudaLaunchConfig_t cfg;
  memset(&cfg, 0, sizeof(cfg));
  cudaLaunchAttribute attr[1];
  cfg.gridDim = grid;
  cfg.blockDim = block;
  cfg.dynamicSmemBytes = smem;
  cfg.stream = stream;
  if (cluster > 0) {
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)cluster; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
  }
  cudaError_t e = cudaLaunchKernelEx(&cfg, kernel, std::forward<Args>(args)...);
  if (e != cudaSuccess) return cuda_fail(e, name);
  g_launches.fetch_add(1, std::memory_order_relaxed);
  t_variant = name;
  return RFIM_OK;
}

// ------------------------------------------------------------------------------------------ TD u8
struct StagedPlan { int nteams, team, slot_bytes, sum_entries, smem; };

bool plan_td_u8_staged(const Call& c, StagedPlan& pl) {
  if (c.window != c.samples) return false;
  // every row must have the same misalignment in src and dst for the aligned interior to match
  if (((reinterpret_cast<uintptr_t>(c.data) ^ reinterpret_cast<uintptr_t>(c.out)) & 15) != 0) return false;
  if (c.samples > 65000) return false;                    // 32-bit S, Q totals inside the kernel
  pl.slot_bytes = (c.samples + 30 + 15) & ~15;
  pl.sum_entries = ((pl.slot_bytes / 16) + 15) & ~15;     // max byte and min byte per 16-byte group
  // per team: one slot, its group summaries, one control block; sixteen teams keep sixteen rows in flight
  const int per_team = pl.slot_bytes + pl.sum_entries * 2 + rfim::kCtrlBytes;
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
  int sms = 0;
  int st = sm_count(sms);
  if (st != RFIM_OK) return st;

  StagedPlan pl;
  const bool can_stage = plan_td_u8_staged(c, pl);
  if (c.variant == 2 && !can_stage) return RFIM_ERR_UNSUPPORTED;
  if (can_stage && c.variant != 1) {
    P.slot_bytes = pl.slot_bytes;
    P.sum_entries = pl.sum_entries;
    const bool med = c.policy == RFIM_REPLACE_MEDIAN;
    if (med && pl.team == 2) return RFIM_ERR_UNSUPPORTED;   // the snapshot median is taken by the one warp that owns the row
    void (*kernel)(const rfim::TdU8Params);
    if (pl.team == 2) kernel = c.flags ? rfim::td_u8_staged_kernel<2, true, false> : rfim::td_u8_staged_kernel<2, false, false>;
    else kernel = c.flags ? (med ? rfim::td_u8_staged_kernel<1, true, true> : rfim::td_u8_staged_kernel<1, true, false>)
                          : (med ? rfim::td_u8_staged_kernel<1, false, true> : rfim::td_u8_staged_kernel<1, false, false>);
    const int threads = pl.nteams * pl.team * 32;
    if ((st = ensure_smem(kernel, (size_t)pl.smem)) != RFIM_OK) return st;
    int occ = 0;
    if ((st = blocks_per_sm(kernel, threads, (size_t)pl.smem, occ)) != RFIM_OK) return st;
    if (occ < 1) occ = 1;
    int64_t grid = (P.rows + pl.nteams - 1) / pl.nteams;
    if (grid > (int64_t)sms * occ) grid = (int64_t)sms * occ;
    if ((st = clear_outputs(c)) != RFIM_OK) return st;
    return launch(med ? "td_u8_staged_median" : (pl.team == 2 ? "td_u8_staged_team2" : "td_u8_staged"),
                  kernel, dim3((unsigned)grid), dim3((unsigned)threads), (size_t)pl.smem, c.stream, 0, P);
  }
  int64_t grid = P.rows;
  if (grid > (int64_t)sms * 32) grid = (int64_t)sms * 32;
  if ((st = clear_outputs(c)) != RFIM_OK) return st;
  return launch("td_u8_generic", rfim::td_u8_generic_kernel, dim3((unsigned)grid), dim3(rfim::kGenericThreads), 0,
                c.stream, 0, P);
}

// ------------------------------------------------------------------------------------------ TD f32
template <int kTW>
int launch_td_f32_t(const Call& c, rfim::TdF32Params& P, bool stage, int sms, const char* name) {
  const int nt = rfim::f32_teams<kTW>();
  const size_t smem = (stage ? (((size_t)P.seg * 4 + 15) & ~(size_t)15) : 0) + (size_t)nt * sizeof(rfim::F32Team) + 16;
  void (*kernel)(const rfim::TdF32Params) = stage ? rfim::td_f32_kernel<kTW, true> : rfim::td_f32_kernel<kTW, false>;
  int st = ensure_smem(kernel, smem);
  if (st != RFIM_OK) return st;
  int occ = 0;
  if ((st = blocks_per_sm(kernel, rfim::kF32Threads, smem, occ)) != RFIM_OK) return st;
  if (occ < 1) return RFIM_ERR_UNSUPPORTED;
  int64_t grid = P.rows * P.segs_per_row;
  if (grid > (int64_t)sms * occ) grid = (int64_t)sms * occ;
  if ((st = clear_outputs(c)) != RFIM_OK) return st;
  return launch(name, kernel, dim3((unsigned)grid), dim3(rfim::kF32Threads), smem, c.stream, 0, P);
}

int launch_td_f32(const Call& c) {
  rfim::TdF32Params P;
  memset(&P, 0, sizeof(P));
  P.src = static_cast<const float*>(c.data);
  P.dst = static_cast<float*>(c.out);
  P.rows = (int64_t)c.beams * c.channels;
  P.stride = c.stride;
  P.S = c.samples;
  P.window = c.window;
  P.n_thr = c.n_thr;
  P.policy = (int)c.policy;
  for (int i = 0; i < c.n_thr; ++i) P.k[i] = c.thr[i];
  P.flags = c.flags;
  P.counts = c.counts;
  int sms = 0;
  int st = sm_count(sms);
  if (st != RFIM_OK) return st;
  // segment = run of whole windows staged in shared memory: the whole row when it fits beside the team
  // scratch with three CTAs per SM, else the whole row alone, else as many windows as fit
  const int overhead = 8 * (int)sizeof(rfim::F32Team) + 16;
  const int cap3 = ((kMaxSmem + 1024) / 3 - 1024 - overhead) / 4;
  const int cap1 = (kMaxSmem - overhead) / 4;
  bool stage = c.variant != 1;
  if (c.samples <= cap1) { P.seg = c.samples; P.segs_per_row = 1; }
  else if (c.window <= cap1) {
    const int cap = c.window <= cap3 ? cap3 : cap1;
    P.seg = cap / c.window * c.window;
    P.segs_per_row = (c.samples + P.seg - 1) / P.seg;
  } else { stage = false; }
  if (!stage) { P.seg = c.samples; P.segs_per_row = 1; }
  if (c.variant == 2 && !stage) return RFIM_ERR_UNSUPPORTED;
  const uintptr_t a = reinterpret_cast<uintptr_t>(c.data) | reinterpret_cast<uintptr_t>(c.out);
  P.bulk = ((a & 15) == 0 && (c.stride % 4 == 0 || P.rows == 1) && (P.segs_per_row == 1 || P.seg % 4 == 0)) ? 1 : 0;
  const int nwin = (P.seg + c.window - 1) / c.window;     // windows per (full) segment
  if (nwin >= 6) return launch_td_f32_t<1>(c, P, stage, sms, stage ? "td_f32_staged_w1" : "td_f32_global_w1");
  if (nwin >= 3) return launch_td_f32_t<2>(c, P, stage, sms, stage ? "td_f32_staged_w2" : "td_f32_global_w2");
  if (nwin == 2) return launch_td_f32_t<4>(c, P, stage, sms, stage ? "td_f32_staged_w4" : "td_f32_global_w4");
  return launch_td_f32_t<8>(c, P, stage, sms, stage ? "td_f32_staged_w8" : "td_f32_global_w8");
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

// One 2-D tensor per 16-byte alignment class k: rows k, k+4, ... of the [rows][pitch] matrix, origin rounded
// down to 16 bytes (off[k] bytes before the row start), box = box_w bytes x box_rows rows.  The last encoding is
// remembered per thread: a real-time caller cleans the same buffers batch after batch.
struct ClassMaps { CUtensorMap m[4]; int off[4]; };
bool encode_class_maps(const uint8_t* base, int64_t stride, int samples, int64_t rows, int box_w, int box_rows,
                       CUtensorMapL2promotion promo, ClassMaps& out) {
  struct Key { const uint8_t* base; int64_t stride; int samples; int64_t rows; int box_w, box_rows, promo; };
  thread_local Key last_key = {nullptr, 0, 0, 0, 0, 0, 0};
  thread_local ClassMaps last_maps;
  Key key;
  memset(&key, 0, sizeof(key));
  key.base = base; key.stride = stride; key.samples = samples; key.rows = rows; key.box_w = box_w;
  key.box_rows = box_rows; key.promo = (int)promo;
  if (last_key.base != nullptr && memcmp(&last_key, &key, sizeof(Key)) == 0) { out = last_maps; return true; }
  EncodeTiledFn enc = encode_tiled_fn();
  if (!enc) return false;
  for (int k = 0; k < 4; ++k) {
    const uintptr_t addr = reinterpret_cast<uintptr_t>(base) + (uintptr_t)k * (uintptr_t)stride;
    out.off[k] = (int)(addr & 15);
    cuuint64_t dims[2] = {(cuuint64_t)samples + (cuuint64_t)out.off[k], (cuuint64_t)(rows / 4)};
    cuuint64_t strides[1] = {(cuuint64_t)4 * (cuuint64_t)stride};
    cuuint32_t box[2] = {(cuuint32_t)box_w, (cuuint32_t)box_rows};
    cuuint32_t estr[2] = {1, 1};
    if (enc(&out.m[k], CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, reinterpret_cast<void*>(addr - out.off[k]), dims, strides,
            box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, promo,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
      return false;
  }
  last_key = key;
  last_maps = out;
  return true;
}

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
  if (encode_tiled_fn() == nullptr) return false;
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

template <int NCH>
int launch_fd_stream_n(const Call& c, const StreamPlan& pl, const rfim::FdStreamMaps& maps,
                       const rfim::FdStreamParams& P, int sms) {
  void (*kernel)(const rfim::FdStreamMaps, const rfim::FdStreamParams);
  const char* name;
  if (pl.binned) {
    kernel = pl.copy ? rfim::fd_u8_stream_kernel<NCH, 3, true, true> : rfim::fd_u8_stream_kernel<NCH, 3, true, false>;
    name = pl.copy ? "fd_u8_stream_binned_copy" : "fd_u8_stream_binned";
  } else {
    kernel = pl.copy ? rfim::fd_u8_stream_kernel<NCH, 4, false, true> : rfim::fd_u8_stream_kernel<NCH, 4, false, false>;
    name = pl.copy ? "fd_u8_stream_copy" : "fd_u8_stream";
  }
  int st = ensure_smem(kernel, (size_t)pl.smem);
  if (st != RFIM_OK) return st;
  int occ = 0;
  if ((st = blocks_per_sm(kernel, rfim::kFsThreads, (size_t)pl.smem, occ)) != RFIM_OK) return st;
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
    void* p = nullptr;
    CUDA_TRY(cudaMallocAsync(&p, 256, c.stream));
    Q.ticket = static_cast<unsigned int*>(p);
    owned = true;
  }
  cudaError_t e = cudaMemsetAsync(Q.ticket, 0, sizeof(unsigned int), c.stream);
  if (e != cudaSuccess) {
    if (owned) cudaFreeAsync(Q.ticket, c.stream);
    return cuda_fail(e, "cudaMemsetAsync(ticket)");
  }
  st = launch(name, kernel, dim3((unsigned)grid), dim3(rfim::kFsThreads), (size_t)pl.smem, c.stream, 0, maps, Q);
  if (owned) {
    e = cudaFreeAsync(Q.ticket, c.stream);
    if (e != cudaSuccess && st == RFIM_OK) st = cuda_fail(e, "cudaFreeAsync(ticket)");
  }
  return st;
}

int launch_fd_stream(const Call& c, const StreamPlan& pl, int sms) {
  rfim::FdStreamParams P;
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
  P.nbins = pl.nbins;
  P.inv_nb = (uint32_t)((((uint64_t)1 << 32) + (uint64_t)P.nb - 1) / (uint64_t)P.nb);
  P.inv_2nb = (uint32_t)((((uint64_t)1 << 32) + 2 * (uint64_t)P.nb - 1) / (2 * (uint64_t)P.nb));
  ClassMaps cm;
  // No L2 promotion: a box row is the 144-byte superset of 128 columns; promoted to whole 128-byte lines it costs
  // two lines (256 bytes) of DRAM traffic, because the half-used line is rarely still in L2 when the neighbouring
  // tile asks for it (measured: 18.2 GB read for a 9.2 GB batch with 128-byte promotion).
  const CUtensorMapL2promotion promo = CU_TENSOR_MAP_L2_PROMOTION_NONE;
  if (!encode_class_maps(P.src, c.stride, c.samples, (int64_t)c.beams * c.channels, rfim::kFsPitchW * 4,
                         rfim::kFsBoxRows, promo, cm))
    return RFIM_ERR_UNSUPPORTED;
  rfim::FdStreamMaps maps;
  for (int k = 0; k < 4; ++k) { maps.src[k] = cm.m[k]; P.off[k] = cm.off[k]; }
  switch (pl.nch) {
    case 4: return launch_fd_stream_n<4>(c, pl, maps, P, sms);
    case 8: return launch_fd_stream_n<8>(c, pl, maps, P, sms);
    case 12: return launch_fd_stream_n<12>(c, pl, maps, P, sms);
    default: return launch_fd_stream_n<16>(c, pl, maps, P, sms);
  }
}

// ---- strip kernel (fd_u8_strip.cuh): all channels x 128 samples per tile resident in shared memory, channels split
// over the smallest cluster whose CTAs fit
struct StripPlan { int cl, rq, smem, box_rows, nw; bool tensor, warp_box; };
// rows per tensor copy: divides the Rq / 4 rows of a class, at most 256, and every box lands 128-byte aligned
int strip_box_rows(int rq) {
  const int rc = rq / 4;
  for (int n = 1; n <= 8; ++n)
    if (rc % n == 0 && rc / n <= 256 && ((rc / n) * rfim::kStripPitchW * 4) % 128 == 0) return rc / n;
  return 0;
}
bool plan_fd_u8_strip(const Call& c, bool want_tensor, int force_cl, StripPlan& pl) {
  if (c.policy != RFIM_REPLACE_MEAN || c.bin_size != c.channels) return false;
  const uintptr_t src = reinterpret_cast<uintptr_t>(c.data), dst = reinterpret_cast<uintptr_t>(c.out);
  if ((src & 3) != 0 || (c.stride & 3) != 0) return false;       // 32-bit word columns
  if (((src ^ dst) & 15) != 0) return false;                     // aligned interiors of src and dst rows coincide
  if (c.channels > 60000) return false;                          // 32-bit column totals inside the kernel
  const size_t half = (size_t)(kMaxSmem + 1024) / 2 - 1024;      // two CTAs per SM (1 KB reserved per CTA)
  // Order of preference (measured on config 4, in place): the whole tile in ONE CTA (one CTA per SM, 32 warps,
  // no cluster barrier) before the smallest cluster whose CTAs fit two to an SM, before the smallest cluster
  // that fits at all.  force_cl: 0 = that order, -1 = skip the single-CTA choice.
  for (int pass = 0; pass < 3; ++pass) {
    for (int cl = 1; cl <= 8; cl *= 2) {
      if (pass == 0 && (cl != 1 || force_cl < 0)) continue;
      if (force_cl > 0 && cl != force_cl) continue;
      const int rq = (c.channels + cl - 1) / cl;
      if (rq > 255 * 16) continue;                               // packed per-thread delta counters (255 rows/thread)
      // tensor copies: every CTA holds whole alignment classes, the rows of a CTA start at a multiple of 4 in the
      // [beams * channels] row index, and every box lands 128-byte aligned in shared memory
      const bool tensor = want_tensor && c.channels % (4 * cl) == 0 && strip_box_rows(rq) > 0 &&
                          encode_tiled_fn() != nullptr;
      const size_t smem = rfim::fd_strip_smem_bytes(rq);
      if (smem > (pass == 1 ? half : (size_t)kMaxSmem)) continue;
      if (pass == 0 && smem <= half) continue;                   // small tiles: two CTAs per SM (pass 1)
      pl.cl = cl; pl.rq = rq; pl.smem = (int)smem; pl.tensor = tensor;
      pl.box_rows = tensor ? strip_box_rows(rq) : 0;
      pl.nw = pass == 1 ? 16 : 32;                               // one CTA per SM: twice the warps
      // one box per warp: Rq / nw consecutive class rows each, 128-byte aligned in shared memory, at most 256
      pl.warp_box = tensor && pl.nw == 32 && rq % (8 * pl.nw) == 0 && rq / pl.nw <= 256;
      if (pl.warp_box) pl.box_rows = rq / pl.nw;
      return true;
    }
  }
  return false;
}

int launch_fd_strip(const Call& c, const StripPlan& pl, int sms) {
  rfim::FdStripParams P;
  memset(&P, 0, sizeof(P));
  P.src = static_cast<const uint8_t*>(c.data);
  P.dst = static_cast<uint8_t*>(c.out);
  P.stride = c.stride;
  P.beams = c.beams; P.C = c.channels; P.S = c.samples;
  P.n_thr = c.n_thr;
  for (int i = 0; i < c.n_thr; ++i) P.p[i] = quantise(c.thr[i]);
  P.flags = c.flags;
  P.counts = c.counts;
  P.Rq = pl.rq;
  P.invC = c.channels >= 2 ? (uint32_t)((((uint64_t)1 << 32) + (uint64_t)c.channels - 1) / (uint64_t)c.channels) : 0u;
  P.tiles_per_beam = (c.samples + rfim::kStripCols - 1) / rfim::kStripCols;
  P.total_tiles = (int64_t)P.tiles_per_beam * c.beams;
  rfim::FdStripMaps maps;
  memset(&maps, 0, sizeof(maps));
  if (pl.tensor) {
    ClassMaps cm;
    if (!encode_class_maps(P.src, c.stride, c.samples, (int64_t)c.beams * c.channels, rfim::kStripPitchW * 4,
                           pl.box_rows, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, cm))
      return RFIM_ERR_UNSUPPORTED;
    for (int k = 0; k < 4; ++k) { maps.src[k] = cm.m[k]; P.off[k] = cm.off[k]; }
    P.box_rows = pl.box_rows;
  }
  auto kernel = pl.nw == 16 ? (pl.tensor ? rfim::fd_u8_strip_kernel<true, 16, false> : rfim::fd_u8_strip_kernel<false, 16, false>)
                : pl.warp_box ? rfim::fd_u8_strip_kernel<true, 32, true>
                              : (pl.tensor ? rfim::fd_u8_strip_kernel<true, 32, false> : rfim::fd_u8_strip_kernel<false, 32, false>);
  int st = ensure_smem(kernel, (size_t)pl.smem);
  if (st != RFIM_OK) return st;
  int nclusters = 0;
  {
    int dev = 0;
    if ((st = current_device(dev)) != RFIM_OK) return st;
    std::lock_guard<std::mutex> lock(g_cache_mutex);
    const auto key = std::make_tuple(dev, reinterpret_cast<const void*>(kernel), 32 * pl.nw, (size_t)pl.smem, pl.cl);
    auto it = g_occupancy.find(key);
    if (it == g_occupancy.end()) {
      cudaLaunchConfig_t cfg;
      memset(&cfg, 0, sizeof(cfg));
      cudaLaunchAttribute attr[1];
      attr[0].id = cudaLaunchAttributeClusterDimension;
      attr[0].val.clusterDim.x = (unsigned)pl.cl; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
      cfg.blockDim = dim3((unsigned)(32 * pl.nw), 1, 1);
      cfg.dynamicSmemBytes = (size_t)pl.smem;
      cfg.attrs = attr;
      cfg.numAttrs = 1;
      cfg.gridDim = dim3((unsigned)(sms * 2 / pl.cl * pl.cl), 1, 1);
      int n = 0;
      CUDA_TRY(cudaOccupancyMaxActiveClusters(&n, kernel, &cfg));
      it = g_occupancy.emplace(key, n).first;
    }
    nclusters = it->second;
  }
  if (nclusters < 1) return RFIM_ERR_UNSUPPORTED;
  int64_t want = P.total_tiles;
  if (want > nclusters) want = nclusters;
  if ((st = clear_outputs(c)) != RFIM_OK) return st;
  static const char* names[2][4] = {{"fd_u8_strip1_bulk", "fd_u8_strip2_bulk", "fd_u8_strip4_bulk", "fd_u8_strip8_bulk"},
                                    {"fd_u8_strip1", "fd_u8_strip2", "fd_u8_strip4", "fd_u8_strip8"}};
  return launch(names[pl.tensor][pl.cl == 1 ? 0 : pl.cl == 2 ? 1 : pl.cl == 4 ? 2 : 3], kernel,
                dim3((unsigned)(want * pl.cl)), dim3((unsigned)(32 * pl.nw)), (size_t)pl.smem, c.stream, pl.cl, maps, P);
}

int launch_fd_u8(const Call& c) {
  int sms = 0;
  int st = sm_count(sms);
  if (st != RFIM_OK) return st;

  // 0 = auto, 2 = any tuned kernel, 16 = the streaming kernel
  if (c.variant == 0 || c.variant == 2 || c.variant == 16) {
    StreamPlan sp;
    if (plan_fd_u8_stream(c, sp)) {
      st = launch_fd_stream(c, sp, sms);
      if (st != RFIM_ERR_UNSUPPORTED) return st;
    }
    if (c.variant == 16) return RFIM_ERR_UNSUPPORTED;
  }
  // 13: strip kernel with per-row bulk copies; 14: never the single-CTA tile; 15: the strip kernel
  if (c.variant == 0 || c.variant == 2 || (c.variant >= 13 && c.variant <= 15)) {
    StripPlan sp;
    if (plan_fd_u8_strip(c, c.variant != 13, c.variant == 14 ? -1 : 0, sp)) {
      st = launch_fd_strip(c, sp, sms);
      if (st != RFIM_ERR_UNSUPPORTED) return st;
    }
  }
  if (c.variant >= 2) return RFIM_ERR_UNSUPPORTED;

  if (c.bin_size != c.channels || c.policy == RFIM_REPLACE_MEDIAN) {   // per-bin mean correction and / or median
    rfim::FdBinnedParams B;                                             // replacement: correctness path
    memset(&B, 0, sizeof(B));
    B.src = static_cast<const uint8_t*>(c.data); B.dst = static_cast<uint8_t*>(c.out); B.stride = c.stride;
    B.beams = c.beams; B.C = c.channels; B.S = c.samples; B.nb = c.bin_size;
    B.n_thr = c.n_thr;
    B.policy = (int)c.policy;
    for (int i = 0; i < c.n_thr; ++i) B.p[i] = quantise(c.thr[i]);
    B.flags = c.flags; B.counts = c.counts;
    const int64_t ncol = (int64_t)c.beams * c.samples;
    int64_t grid = (ncol + rfim::kFdBinnedThreads - 1) / rfim::kFdBinnedThreads;
    if (grid > (int64_t)sms * 16) grid = (int64_t)sms * 16;
    if ((st = clear_outputs(c)) != RFIM_OK) return st;
    return launch("fd_u8_binned_generic", rfim::fd_u8_binned_kernel, dim3((unsigned)grid),
                  dim3(rfim::kFdBinnedThreads), 0, c.stream, 0, B);
  }
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
  const int64_t ncol = (int64_t)c.beams * c.samples;
  int64_t grid = (ncol + rfim::kFdGenericThreads - 1) / rfim::kFdGenericThreads;
  if (grid > (int64_t)sms * 16) grid = (int64_t)sms * 16;
  if ((st = clear_outputs(c)) != RFIM_OK) return st;
  return launch("fd_u8_generic", rfim::fd_u8_generic_kernel, dim3((unsigned)grid), dim3(rfim::kFdGenericThreads), 0,
                c.stream, 0, P);
}

// ------------------------------------------------------------------------------------------ FD f32
int launch_fd_f32(const Call& c) {
  rfim::FdF32Params P;
  memset(&P, 0, sizeof(P));
  P.src = static_cast<const float*>(c.data);
  P.dst = static_cast<float*>(c.out);
  P.stride = c.stride;
  P.beams = c.beams; P.C = c.channels; P.S = c.samples; P.nb = c.bin_size;
  P.n_thr = c.n_thr;
  P.policy = (int)c.policy;
  for (int i = 0; i < c.n_thr; ++i) P.k[i] = c.thr[i];
  P.flags = c.flags;
  P.counts = c.counts;
  if (c.variant >= 2) return RFIM_ERR_UNSUPPORTED;                 // only the correctness path exists
  int sms = 0;
  int st = sm_count(sms);
  if (st != RFIM_OK) return st;
  const int64_t ncol = (int64_t)c.beams * c.samples;
  int64_t grid = (ncol + rfim::kFdF32Threads - 1) / rfim::kFdF32Threads;
  if (grid > (int64_t)sms * 16) grid = (int64_t)sms * 16;
  if ((st = clear_outputs(c)) != RFIM_OK) return st;
  return launch("fd_f32_generic", rfim::fd_f32_generic_kernel, dim3((unsigned)grid), dim3(rfim::kFdF32Threads), 0,
                c.stream, 0, P);
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
  if (variant > 16 || (variant >= 5 && variant <= 12)) return RFIM_ERR_INVALID;
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
