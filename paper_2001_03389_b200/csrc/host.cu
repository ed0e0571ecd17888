// host.cu -- definitions of host.h: error text, per-process caches, tensor-map encoding.
#include "host.h"

#include <atomic>
#include <cmath>
#include <cstdio>
#include <map>
#include <mutex>
#include <tuple>

namespace rfim_host {

std::atomic<uint64_t> g_launches{0};
thread_local char t_cuda_error[256] = "";
thread_local const char* t_variant = "";

int cuda_fail(cudaError_t e, const char* what) {
  snprintf(t_cuda_error, sizeof(t_cuda_error), "%s: %s", what, cudaGetErrorString(e));
  return RFIM_ERR_CUDA;
}
void note_launch(const char* name) {
  g_launches.fetch_add(1, std::memory_order_relaxed);
  t_variant = name;
}
uint64_t launches() { return g_launches.load(std::memory_order_relaxed); }
const char* last_variant() { return t_variant; }
const char* last_cuda_error() { return t_cuda_error; }

namespace {
std::mutex g_cache_mutex;
std::map<std::tuple<int, const void*>, int> g_smem_set;                       // largest opt-in so far
std::map<std::tuple<int, const void*, int, size_t, int>, int> g_occupancy;    // blocks (or clusters) per device
std::map<int, int> g_sms;
}  // namespace

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
int ensure_smem_raw(const void* kernel, size_t bytes) {
  int dev = 0;
  int st = current_device(dev);
  if (st != RFIM_OK) return st;
  std::lock_guard<std::mutex> lock(g_cache_mutex);
  int& have = g_smem_set[std::make_tuple(dev, kernel)];
  if ((int)bytes > have) {
    CUDA_TRY(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
    have = (int)bytes;
  }
  return RFIM_OK;
}
int blocks_per_sm_raw(const void* kernel, int threads, size_t smem, int& occ) {
  int dev = 0;
  int st = current_device(dev);
  if (st != RFIM_OK) return st;
  std::lock_guard<std::mutex> lock(g_cache_mutex);
  const auto key = std::make_tuple(dev, kernel, threads, smem, 0);
  auto it = g_occupancy.find(key);
  if (it == g_occupancy.end()) {
    int n = 0;
    CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, kernel, threads, smem));
    it = g_occupancy.emplace(key, n).first;
  }
  occ = it->second;
  return RFIM_OK;
}
int clusters_per_device_raw(const void* kernel, int threads, size_t smem, int cluster, int sms, int& n_out) {
  int dev = 0;
  int st = current_device(dev);
  if (st != RFIM_OK) return st;
  std::lock_guard<std::mutex> lock(g_cache_mutex);
  const auto key = std::make_tuple(dev, kernel, threads, smem, cluster);
  auto it = g_occupancy.find(key);
  if (it == g_occupancy.end()) {
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)cluster; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.blockDim = dim3((unsigned)threads, 1, 1);
    cfg.dynamicSmemBytes = smem;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    cfg.gridDim = dim3((unsigned)(sms * 2 / cluster * cluster), 1, 1);
    int n = 0;
    CUDA_TRY(cudaOccupancyMaxActiveClusters(&n, kernel, &cfg));
    it = g_occupancy.emplace(key, n).first;
  }
  n_out = it->second;
  return RFIM_OK;
}

uint32_t quantise(double k) { return (uint32_t)std::nearbyint(k * 65536.0); }

int clear_outputs(const Call& c) {
  if (c.keep_outputs) return RFIM_OK;
  if (c.flags)
    CUDA_TRY(cudaMemsetAsync(c.flags, 0, (size_t)c.beams * c.channels * c.samples, c.stream));
  if (c.counts && c.n_thr > 0)
    CUDA_TRY(cudaMemsetAsync(c.counts, 0, sizeof(unsigned long long) * c.n_thr, c.stream));
  return RFIM_OK;
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static EncodeTiledFn encode_tiled_fn() {
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
bool tensor_maps_available() { return encode_tiled_fn() != nullptr; }

bool encode_class_maps(const uint8_t* base, int64_t stride, int samples, int64_t rows, int box_w, int box_rows,
                       CUtensorMapL2promotion promo, ClassMaps& out) {
  struct Key { const uint8_t* base; int64_t stride; int samples; int64_t rows; int box_w, box_rows, promo; };
  // the two most recent encodings are remembered (a source and a destination buffer per call)
  thread_local Key last_key[2] = {{nullptr, 0, 0, 0, 0, 0, 0}, {nullptr, 0, 0, 0, 0, 0, 0}};
  thread_local ClassMaps last_maps[2];
  thread_local int next_slot = 0;
  Key key;
  memset(&key, 0, sizeof(key));
  key.base = base; key.stride = stride; key.samples = samples; key.rows = rows; key.box_w = box_w;
  key.box_rows = box_rows; key.promo = (int)promo;
  for (int i = 0; i < 2; ++i)
    if (last_key[i].base != nullptr && memcmp(&last_key[i], &key, sizeof(Key)) == 0) { out = last_maps[i]; return true; }
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
  last_key[next_slot] = key;
  last_maps[next_slot] = out;
  next_slot ^= 1;
  return true;
}

bool encode_f32_map(const float* base, int64_t pitch_bytes, int cols, int64_t rows, int box_cols, int box_rows,
                    CUtensorMap& out) {
  EncodeTiledFn enc = encode_tiled_fn();
  if (!enc) return false;
  cuuint64_t dims[2] = {(cuuint64_t)cols, (cuuint64_t)rows};
  cuuint64_t strides[1] = {(cuuint64_t)pitch_bytes};
  cuuint32_t box[2] = {(cuuint32_t)box_cols, (cuuint32_t)box_rows};
  cuuint32_t estr[2] = {1, 1};
  return enc(&out, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<float*>(base), dims, strides, box, estr,
             CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
             CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

}  // namespace rfim_host
