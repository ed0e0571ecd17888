// rfim_api.cu -- the C ABI of librfim (include/rfim.h): argument checks, variant selection,
// launches.  No CPU fallback: every step of the path runs in the kernels of this directory.
#include "../../include/rfim.h"

#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstring>

#include "common.cuh"
#include "fd_u8.cuh"
#include "fd_f32.cuh"
#include "fd_u8_binned.cuh"
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
  if (z.variant < 0 || z.variant > 14) return RFIM_ERR_INVALID;
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
struct StagedPlan { int nteams, team, slot_bytes, sum_entries, smem; };

bool plan_td_u8_staged(const Call& c, StagedPlan& pl) {
  if (c.window != c.samples || c.policy != RFIM_REPLACE_MEAN) return false;
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
  DevInfo dv;
  int st = dev_info(dv);
  if (st != RFIM_OK) return st;

  StagedPlan pl;
  const bool can_stage = plan_td_u8_staged(c, pl);
  if (c.variant == 2 && !can_stage) return RFIM_ERR_UNSUPPORTED;
  if (can_stage && c.variant != 1) {
    P.slot_bytes = pl.slot_bytes;
    P.sum_entries = pl.sum_entries;
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


// ------------------------------------------------------------------------------------------ TD f32
template <int kTW>
int launch_td_f32_t(const Call& c, rfim::TdF32Params& P, bool stage, int sms, const char* name) {
  const int nt = rfim::f32_teams<kTW>();
  const size_t smem = (stage ? (((size_t)P.seg * 4 + 15) & ~(size_t)15) : 0) + (size_t)nt * sizeof(rfim::F32Team) + 16;
  void (*kernel)(const rfim::TdF32Params) = stage ? rfim::td_f32_kernel<kTW, true> : rfim::td_f32_kernel<kTW, false>;
  CUDA_TRY(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  int occ = 0;
  CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kernel, rfim::kF32Threads, smem));
  if (occ < 1) return RFIM_ERR_UNSUPPORTED;
  int64_t grid = P.rows * P.segs_per_row;
  if (grid > (int64_t)sms * occ) grid = (int64_t)sms * occ;
  int st = clear_outputs(c);
  if (st != RFIM_OK) return st;
  kernel<<<(unsigned)grid, rfim::kF32Threads, smem, c.stream>>>(P);
  return after_launch(name);
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
  DevInfo dv;
  int st = dev_info(dv);
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
  if (nwin >= 6) return launch_td_f32_t<1>(c, P, stage, dv.sms, stage ? "td_f32_staged_w1" : "td_f32_global_w1");
  if (nwin >= 3) return launch_td_f32_t<2>(c, P, stage, dv.sms, stage ? "td_f32_staged_w2" : "td_f32_global_w2");
  if (nwin == 2) return launch_td_f32_t<4>(c, P, stage, dv.sms, stage ? "td_f32_staged_w4" : "td_f32_global_w4");
  return launch_td_f32_t<8>(c, P, stage, dv.sms, stage ? "td_f32_staged_w8" : "td_f32_global_w8");
}

// ------------------------------------------------------------------------------------------ FD u8
// Geometry of the cluster kernel for the request, or false when only the generic kernel can run it.
struct FdPlan { int cl, pw, ts, wc, rq, rg, tiles_per_beam, smem; };

constexpr int kFdPw[] = {136, 120, 104, 88, 72, 56, 40, 24};    // row pitches (words), PW mod 32 in {8, 24}

bool plan_fd_u8_for(const Call& c, int cl, int rg, size_t budget, FdPlan& pl) {
  const int rq = (c.channels + cl - 1) / cl;
  if (rq > 255 * rg) return false;                               // packed per-thread delta counters (255 rows/thread)
  if (rg == 1 && cl < 4) return false;                           // column owners: 4 * ceil(WC / cl) threads <= WC
  for (int pw : kFdPw) {
    int ts_max = 4 * pw - 16;
    if (ts_max > 512) ts_max = 512;                              // 4 * WC <= 512 threads
    const int tiles = (c.samples + ts_max - 1) / ts_max;
    int ts = (c.samples + tiles - 1) / tiles;
    ts = (ts + 3) & ~3;
    const int wc = rg == 1 ? ((ts / 4) + 31) & ~31 : ((ts / 4) + 7) & ~7;   // blockDim = rg * wc, whole warps
    const size_t smem = rfim::fd_cluster_smem_bytes(pw, rq, wc);
    if (smem > budget) continue;
    pl.cl = cl; pl.pw = pw; pl.ts = ts; pl.wc = wc; pl.rq = rq; pl.rg = rg; pl.tiles_per_beam = tiles; pl.smem = (int)smem;
    return true;
  }
  return false;
}

bool plan_fd_u8_cluster(const Call& c, int force_cl, int rg, FdPlan& pl) {
  if (c.policy != RFIM_REPLACE_MEAN || c.bin_size != c.channels) return false;
  const uintptr_t src = reinterpret_cast<uintptr_t>(c.data), dst = reinterpret_cast<uintptr_t>(c.out);
  if ((src & 3) != 0 || (c.stride & 3) != 0) return false;       // 32-bit word columns
  if (((src ^ dst) & 15) != 0) return false;                     // aligned interiors of src and dst rows coincide
  if (c.channels > 60000) return false;                          // 32-bit column totals inside the kernel
  const size_t half = (size_t)(kMaxSmem + 1024) / 2 - 1024;      // two CTAs per SM (1 KB reserved per CTA)
  if (force_cl) return plan_fd_u8_for(c, force_cl, rg, half, pl) || plan_fd_u8_for(c, force_cl, rg, (size_t)kMaxSmem, pl);
  // smallest cluster that still gets the widest tile with two CTAs per SM; else the widest tile any cluster gets
  FdPlan best; bool have = false;
  for (int cl = 1; cl <= 8; cl *= 2) {
    FdPlan p;
    if (!plan_fd_u8_for(c, cl, rg, half, p)) continue;
    if (!have || p.ts > best.ts) { best = p; have = true; }
    if (p.pw == kFdPw[0]) break;
  }
  if (!have) {
    for (int cl = 8; cl >= 1 && !have; cl /= 2) have = plan_fd_u8_for(c, cl, rg, (size_t)kMaxSmem, best);
  }
  if (have) pl = best;
  return have;
}

template <int PW, int RG>
int launch_fd_cluster_rg(const Call& c, const FdPlan& pl, const rfim::FdU8Params& P, int sms) {
  auto kernel = rfim::fd_u8_cluster_kernel<PW, RG>;
  CUDA_TRY(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, pl.smem));
  cudaLaunchConfig_t cfg;
  memset(&cfg, 0, sizeof(cfg));
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = (unsigned)pl.cl; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
  cfg.blockDim = dim3((unsigned)(RG * pl.wc), 1, 1);
  cfg.dynamicSmemBytes = (size_t)pl.smem;
  cfg.stream = c.stream;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  int nclusters = 0;
  cfg.gridDim = dim3((unsigned)(sms * 2 / pl.cl * pl.cl), 1, 1);
  CUDA_TRY(cudaOccupancyMaxActiveClusters(&nclusters, kernel, &cfg));
  if (nclusters < 1) return RFIM_ERR_UNSUPPORTED;
  int64_t want = P.total_tiles;
  if (want > nclusters) want = nclusters;
  cfg.gridDim = dim3((unsigned)(want * pl.cl), 1, 1);
  int st = clear_outputs(c);
  if (st != RFIM_OK) return st;
  CUDA_TRY(cudaLaunchKernelEx(&cfg, kernel, P));
  static const char* names[2][4] = {{"fd_u8_cluster1", "fd_u8_cluster2", "fd_u8_cluster4", "fd_u8_cluster8"},
                                    {"fd_u8_cluster1_rg1", "fd_u8_cluster2_rg1", "fd_u8_cluster4_rg1", "fd_u8_cluster8_rg1"}};
  return after_launch(names[RG == 1][pl.cl == 1 ? 0 : pl.cl == 2 ? 1 : pl.cl == 4 ? 2 : 3]);
}
template <int PW>
int launch_fd_cluster(const Call& c, const FdPlan& pl, const rfim::FdU8Params& P, int sms) {
  return pl.rg == 1 ? launch_fd_cluster_rg<PW, 1>(c, pl, P, sms) : launch_fd_cluster_rg<PW, 4>(c, pl, P, sms);
}

// strip kernel: all channels x 128 samples per tile, channels split over the smallest cluster whose CTAs fit
// two to an SM (else one to an SM)
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

// one 2-D tensor per 16-byte alignment class k: rows k, k+4, ... of the [beams*channels][pitch] matrix, origin
// rounded down to 16 bytes (off[k] bytes before the row start), box = 128 bytes x (channels per CTA) / 4 rows
bool encode_strip_maps(const Call& c, uint8_t* base, int box_rows, CUtensorMap* maps, int* off) {
  EncodeTiledFn enc = encode_tiled_fn();
  if (!enc) return false;
  for (int k = 0; k < 4; ++k) {
    const uintptr_t addr = reinterpret_cast<uintptr_t>(base) + (uintptr_t)k * (uintptr_t)c.stride;
    off[k] = (int)(addr & 15);
    cuuint64_t dims[2] = {(cuuint64_t)c.samples + (cuuint64_t)off[k], (cuuint64_t)c.beams * (cuuint64_t)c.channels / 4};
    cuuint64_t strides[1] = {(cuuint64_t)4 * (cuuint64_t)c.stride};
    cuuint32_t box[2] = {(cuuint32_t)(rfim::kStripPitchW * 4), (cuuint32_t)box_rows};
    cuuint32_t estr[2] = {1, 1};
    if (enc(&maps[k], CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, reinterpret_cast<void*>(addr - off[k]), dims, strides, box,
            estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
      return false;
  }
  return true;
}

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
  // no cluster barrier: 6.7 ms) before the smallest cluster whose CTAs fit two to an SM (7.1 ms with two CTAs),
  // before the smallest cluster that fits at all.  force_cl: 0 = that order, -1 = skip the single-CTA choice.
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
    if (!encode_strip_maps(c, const_cast<uint8_t*>(P.src), pl.box_rows, maps.src, P.off)) return RFIM_ERR_UNSUPPORTED;
    P.box_rows = pl.box_rows;
  }
  auto kernel = pl.nw == 16 ? (pl.tensor ? rfim::fd_u8_strip_kernel<true, 16, false> : rfim::fd_u8_strip_kernel<false, 16, false>)
                : pl.warp_box ? rfim::fd_u8_strip_kernel<true, 32, true>
                              : (pl.tensor ? rfim::fd_u8_strip_kernel<true, 32, false> : rfim::fd_u8_strip_kernel<false, 32, false>);
  CUDA_TRY(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, pl.smem));
  cudaLaunchConfig_t cfg;
  memset(&cfg, 0, sizeof(cfg));
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = (unsigned)pl.cl; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
  cfg.blockDim = dim3((unsigned)(32 * pl.nw), 1, 1);
  cfg.dynamicSmemBytes = (size_t)pl.smem;
  cfg.stream = c.stream;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  int nclusters = 0;
  cfg.gridDim = dim3((unsigned)(sms * 2 / pl.cl * pl.cl), 1, 1);
  CUDA_TRY(cudaOccupancyMaxActiveClusters(&nclusters, kernel, &cfg));
  if (nclusters < 1) return RFIM_ERR_UNSUPPORTED;
  int64_t want = P.total_tiles;
  if (want > nclusters) want = nclusters;
  cfg.gridDim = dim3((unsigned)(want * pl.cl), 1, 1);
  int st = clear_outputs(c);
  if (st != RFIM_OK) return st;
  CUDA_TRY(cudaLaunchKernelEx(&cfg, kernel, maps, P));
  static const char* names[2][4] = {{"fd_u8_strip1_bulk", "fd_u8_strip2_bulk", "fd_u8_strip4_bulk", "fd_u8_strip8_bulk"},
                                    {"fd_u8_strip1", "fd_u8_strip2", "fd_u8_strip4", "fd_u8_strip8"}};
  return after_launch(names[pl.tensor][pl.cl == 1 ? 0 : pl.cl == 2 ? 1 : pl.cl == 4 ? 2 : 3]);
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

  if (c.bin_size != c.channels || c.policy == RFIM_REPLACE_MEDIAN) {   // per-bin mean correction and / or median
    if (c.variant >= 2) return RFIM_ERR_UNSUPPORTED;                    // replacement: correctness path
    rfim::FdBinnedParams B;
    memset(&B, 0, sizeof(B));
    B.src = P.src; B.dst = P.dst; B.stride = c.stride;
    B.beams = c.beams; B.C = c.channels; B.S = c.samples; B.nb = c.bin_size;
    B.n_thr = c.n_thr;
    B.policy = (int)c.policy;
    for (int i = 0; i < c.n_thr; ++i) B.p[i] = P.p[i];
    B.flags = c.flags; B.counts = c.counts;
    const int64_t ncol = (int64_t)c.beams * c.samples;
    int64_t grid = (ncol + rfim::kFdBinnedThreads - 1) / rfim::kFdBinnedThreads;
    if (grid > (int64_t)dv.sms * 16) grid = (int64_t)dv.sms * 16;
    if ((st = clear_outputs(c)) != RFIM_OK) return st;
    rfim::fd_u8_binned_kernel<<<(unsigned)grid, rfim::kFdBinnedThreads, 0, c.stream>>>(B);
    return after_launch("fd_u8_binned_generic");
  }

  if (c.variant == 0 || c.variant == 2 || c.variant == 13 || c.variant == 14) {
    // 13: strip kernel with per-row bulk copies; 14: never the single-CTA tile (clusters, two CTAs per SM)
    StripPlan sp;
    if (plan_fd_u8_strip(c, c.variant != 13, c.variant == 14 ? -1 : 0, sp)) {
      st = launch_fd_strip(c, sp, dv.sms);
      if (st != RFIM_ERR_UNSUPPORTED) return st;
    }
  }
  FdPlan pl;
  int force_cl = 0, rg = 4;
  if (c.variant >= 5 && c.variant <= 8) force_cl = 1 << (c.variant - 5);
  if (c.variant >= 9 && c.variant <= 12) { force_cl = 1 << (c.variant - 9); rg = 1; }
  const bool can_cluster = c.variant != 1 && plan_fd_u8_cluster(c, force_cl, rg, pl);
  if (c.variant >= 2 && !can_cluster) return RFIM_ERR_UNSUPPORTED;
  if (can_cluster) {
    P.Ts = pl.ts; P.WC = pl.wc; P.Rq = pl.rq;
    P.tiles_per_beam = pl.tiles_per_beam;
    P.total_tiles = (int64_t)pl.tiles_per_beam * c.beams;
    switch (pl.pw) {
      case 136: st = launch_fd_cluster<136>(c, pl, P, dv.sms); break;
      case 120: st = launch_fd_cluster<120>(c, pl, P, dv.sms); break;
      case 104: st = launch_fd_cluster<104>(c, pl, P, dv.sms); break;
      case 88: st = launch_fd_cluster<88>(c, pl, P, dv.sms); break;
      case 72: st = launch_fd_cluster<72>(c, pl, P, dv.sms); break;
      case 56: st = launch_fd_cluster<56>(c, pl, P, dv.sms); break;
      case 40: st = launch_fd_cluster<40>(c, pl, P, dv.sms); break;
      default: st = launch_fd_cluster<24>(c, pl, P, dv.sms); break;
    }
    if (st != RFIM_ERR_UNSUPPORTED || c.variant >= 2) return st;
  }
  if (c.policy != RFIM_REPLACE_MEAN || c.bin_size != c.channels) return RFIM_ERR_UNSUPPORTED;
  const int64_t ncol = (int64_t)c.beams * c.samples;
  int64_t grid = (ncol + rfim::kFdGenericThreads - 1) / rfim::kFdGenericThreads;
  if (grid > (int64_t)dv.sms * 16) grid = (int64_t)dv.sms * 16;
  if ((st = clear_outputs(c)) != RFIM_OK) return st;
  rfim::fd_u8_generic_kernel<<<(unsigned)grid, rfim::kFdGenericThreads, 0, c.stream>>>(P);
  return after_launch("fd_u8_generic");
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
  DevInfo dv;
  int st = dev_info(dv);
  if (st != RFIM_OK) return st;
  const int64_t ncol = (int64_t)c.beams * c.samples;
  int64_t grid = (ncol + rfim::kFdF32Threads - 1) / rfim::kFdF32Threads;
  if (grid > (int64_t)dv.sms * 16) grid = (int64_t)dv.sms * 16;
  if ((st = clear_outputs(c)) != RFIM_OK) return st;
  rfim::fd_f32_generic_kernel<<<(unsigned)grid, rfim::kFdF32Threads, 0, c.stream>>>(P);
  return after_launch("fd_f32_generic");
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
  return launch_td_f32(c);
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
  return launch_fd_f32(c);
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
    // dense rows: one linear copy (a 2-D copy of 12500-byte rows is markedly slower over PCIe)
    cudaError_t e = stride == samples
                        ? cudaMemcpyAsync(dev[slot], h_in, rows * (size_t)samples * es, cudaMemcpyHostToDevice, streams[slot])
                        : cudaMemcpy2DAsync(dev[slot], (size_t)stride * es, h_in, (size_t)stride * es,
                                            (size_t)samples * es, rows, cudaMemcpyHostToDevice, streams[slot]);
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
    e = stride == samples
            ? cudaMemcpyAsync(h_out, dev[slot], rows * (size_t)samples * es, cudaMemcpyDeviceToHost, streams[slot])
            : cudaMemcpy2DAsync(h_out, (size_t)stride * es, dev[slot], (size_t)stride * es, (size_t)samples * es, rows,
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
