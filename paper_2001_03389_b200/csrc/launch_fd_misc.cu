// launch_fd_misc.cu -- variant selection over the FDSC uint8 kernel families, and the launches of the correctness
// paths (fd_u8.cuh, fd_u8_binned.cuh, fd_f32.cuh).
#include "host.h"
#include "fd_u8.cuh"
#include "fd_f32.cuh"
#include "fd_f32_tile.cuh"
#include "fd_f32_bins.cuh"
#include "fd_u8_binned.cuh"

namespace rfim_host {

int launch_fd_u8(const Call& c) {
  int sms = 0;
  int st = sm_count(sms);
  if (st != RFIM_OK) return st;

  // 0 = auto, 2 = any tuned kernel, 16 = the streaming kernel, 17 = the class-per-warp streaming kernel, 18 = its
  // binned form.
  // Auto order (measured on B200 on raw config-3 / config-4 data).  One bin, in place: the resident-
  // tile strip kernel for short batches (12 beams: 0.153 ms vs 0.170), the class-per-warp streaming kernel from about
  // 40 beams on (96 beams: 0.93 ms vs 1.07; 240 beams: 2.21 vs 2.61).  Out of place the strip kernel copies the tile
  // while its statistics pass reads it and stays ahead until about 200 beams (96 beams: 1.28 ms vs 1.89; 240: 4.48
  // vs 4.62; 480: 10.2 vs 9.2).  Bins -> one streaming pass per threshold step (fd_u8_qbin.cuh).
  const bool one_bin = c.bin_size == c.channels;
  const bool tuned = c.variant == 0 || c.variant == 2;
  const int64_t tiles = (int64_t)c.beams * ((c.samples + 127) / 128);
  if (tuned && one_bin && tiles < (c.out != c.data ? 20000 : 4000)) {
    st = try_fd_u8_strip(c, true, 0, sms);
    if (st != RFIM_ERR_UNSUPPORTED) return st;
  }
  if (tuned || c.variant == 17) {
    st = try_fd_u8_quad(c, sms);
    if (st != RFIM_ERR_UNSUPPORTED || c.variant == 17) return st;
  }
  if (tuned || c.variant == 18) {                     // bins: pooled repair (96 beams, bins of 32: see DESIGN.md 6.2c)
    st = try_fd_u8_qbin(c, sms);
    if (st != RFIM_ERR_UNSUPPORTED || c.variant == 18) return st;
  }
  if (tuned || c.variant == 16) {
    st = try_fd_u8_stream(c, sms);
    if (st != RFIM_ERR_UNSUPPORTED) return st;
    if (c.variant == 16) return RFIM_ERR_UNSUPPORTED;
  }
  // 13: strip kernel with per-row bulk copies; 14: never the single-CTA tile; 15: the strip kernel
  if (c.variant == 0 || c.variant == 2 || (c.variant >= 13 && c.variant <= 15)) {
    st = try_fd_u8_strip(c, c.variant != 13, c.variant == 14 ? -1 : 0, sms);
    if (st != RFIM_ERR_UNSUPPORTED) return st;
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
// the resident-tile kernel (fd_f32_tile.cuh): one bin, all channels x 32 samples per tile in shared memory
int try_fd_f32_tile(const Call& c, int sms) {
  const bool binned = c.bin_size != c.channels;                                 // fd_f32_bins.cuh: a thread owns whole bins
  if (binned && c.bin_size > 64) return RFIM_ERR_UNSUPPORTED;                   // (one 64-bit flag word per bin)
  const uintptr_t a = reinterpret_cast<uintptr_t>(c.data) | reinterpret_cast<uintptr_t>(c.out);
  if ((a & 15) != 0 || c.stride % 4 != 0) return RFIM_ERR_UNSUPPORTED;          // tensor maps: 16-byte pitch and base
  if (c.channels < 2 || c.channels > 32768) return RFIM_ERR_UNSUPPORTED;
  // tiles of 16 samples when two CTAs then fit an SM (their loads, sweeps and stores overlap), else 32
  const size_t half = (size_t)(kMaxSmem + 1024) / 2 - 1024;
  const bool narrow = rfim::fd_f32_tile_smem_bytes<16>(c.channels) <= half;
  const int cols = narrow ? 16 : 32;
  const size_t smem = narrow ? rfim::fd_f32_tile_smem_bytes<16>(c.channels) : rfim::fd_f32_tile_smem_bytes<32>(c.channels);
  if (smem > (size_t)kMaxSmem) return RFIM_ERR_UNSUPPORTED;
  if (!tensor_maps_available()) return RFIM_ERR_UNSUPPORTED;
  int box_rows = 0;                                                            // largest divisor of C up to 256
  for (int d = 256; d >= 1; --d)
    if (c.channels % d == 0) { box_rows = d; break; }
  const int nboxes = c.channels / box_rows;
  if (nboxes > rfim::kFtMaxBoxes) return RFIM_ERR_UNSUPPORTED;
  if ((int64_t)c.beams * c.channels > 0x7fffffff) return RFIM_ERR_UNSUPPORTED;  // tensor coordinates
  rfim::FdF32TileParams P;
  memset(&P, 0, sizeof(P));
  P.src = static_cast<const float*>(c.data);
  P.dst = static_cast<float*>(c.out);
  P.stride = c.stride;
  P.beams = c.beams; P.C = c.channels; P.S = c.samples;
  P.n_thr = c.n_thr;
  P.policy = (int)c.policy;
  for (int i = 0; i < c.n_thr; ++i) P.k[i] = c.thr[i];
  P.flags = c.flags;
  P.counts = c.counts;
  P.box_rows = box_rows; P.nboxes = nboxes;
  P.tiles_per_beam = (c.samples + cols - 1) / cols;
  P.total_tiles = (int64_t)P.tiles_per_beam * c.beams;
  P.copy = c.out != c.data ? 1 : 0;
  rfim::FdF32TileMaps maps;
  memset(&maps, 0, sizeof(maps));
  const int64_t rows = (int64_t)c.beams * c.channels;
  if (!encode_f32_map(P.src, c.stride * 4, c.samples, rows, cols, box_rows, maps.src)) return RFIM_ERR_UNSUPPORTED;
  if (!encode_f32_map(P.dst, c.stride * 4, c.samples, rows, cols, box_rows, maps.dst)) return RFIM_ERR_UNSUPPORTED;
  if (binned) {
    auto bkernel = narrow ? rfim::fd_f32_bins_kernel<16> : rfim::fd_f32_bins_kernel<32>;
    int st = ensure_smem(bkernel, smem);
    if (st != RFIM_OK) return st;
    int occ = 0;
    if ((st = blocks_per_sm(bkernel, rfim::kFtThreads, smem, occ)) != RFIM_OK) return st;
    if (occ < 1) return RFIM_ERR_UNSUPPORTED;
    int64_t grid = P.total_tiles;
    if (grid > (int64_t)sms * occ) grid = (int64_t)sms * occ;
    if ((st = clear_outputs(c)) != RFIM_OK) return st;
    return launch(P.policy ? "fd_f32_bins_median" : "fd_f32_bins", bkernel, dim3((unsigned)grid), dim3(rfim::kFtThreads),
                  smem, c.stream, 0, maps, P, c.bin_size);
  }
  auto kernel = narrow ? rfim::fd_f32_tile_kernel<16> : rfim::fd_f32_tile_kernel<32>;
  int st = ensure_smem(kernel, smem);
  if (st != RFIM_OK) return st;
  int occ = 0;
  if ((st = blocks_per_sm(kernel, rfim::kFtThreads, smem, occ)) != RFIM_OK) return st;
  if (occ < 1) return RFIM_ERR_UNSUPPORTED;
  int64_t grid = P.total_tiles;
  if (grid > (int64_t)sms * occ) grid = (int64_t)sms * occ;
  if ((st = clear_outputs(c)) != RFIM_OK) return st;
  return launch(P.policy ? "fd_f32_tile_median" : "fd_f32_tile", kernel, dim3((unsigned)grid), dim3(rfim::kFtThreads),
                smem, c.stream, 0, maps, P);
}

int launch_fd_f32(const Call& c) {
  if (c.variant == 0 || c.variant == 2) {
    int sms0 = 0;
    int st0 = sm_count(sms0);
    if (st0 != RFIM_OK) return st0;
    st0 = try_fd_f32_tile(c, sms0);
    if (st0 != RFIM_ERR_UNSUPPORTED) return st0;
  }
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

}  // namespace rfim_host
