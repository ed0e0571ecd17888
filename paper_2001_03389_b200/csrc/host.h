// host.h -- host-side plumbing shared by the launch units of librfim (one translation unit per kernel family, so
// that the families compile in parallel): the validated call, per-process caches of launch attributes, the launch
// wrapper, tensor-map encoding.  Nothing here touches the data.
#pragma once

#include "../../include/rfim.h"

#include <cuda.h>
#include <cuda_runtime.h>

#include <cstdint>
#include <cstring>
#include <utility>

namespace rfim_host {

constexpr int kMaxSmem = 227 * 1024;   // opt-in dynamic shared memory per CTA on sm_100

int cuda_fail(cudaError_t e, const char* what);
#define CUDA_TRY(expr)                                              \
  do {                                                              \
    cudaError_t e_ = (expr);                                        \
    if (e_ != cudaSuccess) return ::rfim_host::cuda_fail(e_, #expr); \
  } while (0)

int current_device(int& dev);
int sm_count(int& sms);
// Launch attributes do not depend on the data: shared-memory opt-in and occupancy are set / queried once per
// (device, kernel, block size, shared memory) and remembered, so a small real-time call (12 beams, ~0.1 ms)
// pays for the launch only.
int ensure_smem_raw(const void* kernel, size_t bytes);
int blocks_per_sm_raw(const void* kernel, int threads, size_t smem, int& occ);
int clusters_per_device_raw(const void* kernel, int threads, size_t smem, int cluster, int sms, int& n);
template <typename K>
int ensure_smem(K kernel, size_t bytes) { return ensure_smem_raw(reinterpret_cast<const void*>(kernel), bytes); }
// resident CTAs per SM of a plain (non-cluster) kernel
template <typename K>
int blocks_per_sm(K kernel, int threads, size_t smem, int& occ) {
  return blocks_per_sm_raw(reinterpret_cast<const void*>(kernel), threads, smem, occ);
}

inline size_t elem_size(rfim_dtype t) { return t == RFIM_U8 ? 1 : 4; }
// p = round-half-even(k * 2^16): k * 65536 is exact, nearbyint rounds half to even (default mode)
uint32_t quantise(double k);

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

// flags / counts are defined as "overwritten": clear them on the stream before the kernel adds to them
int clear_outputs(const Call& c);
void note_launch(const char* name);

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
  note_launch(name);
  return RFIM_OK;
}

// One 2-D tensor per 16-byte alignment class k: rows k, k+4, ... of the [rows][pitch] matrix, origin rounded
// down to 16 bytes (off[k] bytes before the row start), box = box_w bytes x box_rows rows.  The last encoding is
// remembered per thread: a real-time caller cleans the same buffers batch after batch.
struct ClassMaps { CUtensorMap m[4]; int off[4]; };
bool tensor_maps_available();
bool encode_class_maps(const uint8_t* base, int64_t stride, int samples, int64_t rows, int box_w, int box_rows,
                       CUtensorMapL2promotion promo, ClassMaps& out);

// a plain 2-D tensor map over [rows][cols] float32 with row pitch `pitch_bytes` (a multiple of 16, base 16-byte
// aligned), box = box_cols x box_rows elements
bool encode_f32_map(const float* base, int64_t pitch_bytes, int cols, int64_t rows, int box_cols, int box_rows,
                    CUtensorMap& out);

// the launch units (each returns an rfim_status; RFIM_ERR_UNSUPPORTED = no kernel of that family takes the call)
int launch_td_u8(const Call& c);
int launch_td_f32(const Call& c);
int launch_fd_u8(const Call& c);          // launch_fd_misc.cu: variant selection over the FDSC u8 families
int launch_fd_f32(const Call& c);
int try_fd_u8_stream(const Call& c, int sms);                              // launch_fd_stream.cu
int try_fd_u8_quad(const Call& c, int sms);                                // launch_fd_stream.cu
int try_fd_u8_qbin(const Call& c, int sms);                                // launch_fd_stream.cu
int try_fd_u8_strip(const Call& c, bool want_tensor, int force_cl, int sms);   // launch_fd_strip.cu

}  // namespace rfim_host
