// launch_fd_strip.cu -- geometry and launch of the resident-tile FDSC uint8 kernel (fd_u8_strip.cuh).
#include "host.h"
#include "fd_u8_strip.cuh"

namespace rfim_host {

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
  if (c.bin_size != c.channels) return false;
  const bool median = c.policy == RFIM_REPLACE_MEDIAN;           // the median search runs inside ONE CTA per tile
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
      if (median && cl != 1) continue;
      const int rq = (c.channels + cl - 1) / cl;
      if (rq > 255 * 16) continue;                               // packed per-thread delta counters (255 rows/thread)
      // tensor copies: every CTA holds whole alignment classes, the rows of a CTA start at a multiple of 4 in the
      // [beams * channels] row index, and every box lands 128-byte aligned in shared memory
      const bool tensor = want_tensor && c.channels % (4 * cl) == 0 && strip_box_rows(rq) > 0 &&
                          tensor_maps_available();
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
  const bool median = c.policy == RFIM_REPLACE_MEDIAN;
  auto kernel = pl.nw == 16 ? (pl.tensor ? rfim::fd_u8_strip_kernel<true, 16, false> : rfim::fd_u8_strip_kernel<false, 16, false>)
                : pl.warp_box ? rfim::fd_u8_strip_kernel<true, 32, true>
                              : (pl.tensor ? rfim::fd_u8_strip_kernel<true, 32, false> : rfim::fd_u8_strip_kernel<false, 32, false>);
  if (median)
    kernel = pl.nw == 16 ? (pl.tensor ? rfim::fd_u8_strip_kernel<true, 16, false, true> : rfim::fd_u8_strip_kernel<false, 16, false, true>)
             : pl.warp_box ? rfim::fd_u8_strip_kernel<true, 32, true, true>
                           : (pl.tensor ? rfim::fd_u8_strip_kernel<true, 32, false, true> : rfim::fd_u8_strip_kernel<false, 32, false, true>);
  int st = ensure_smem(kernel, (size_t)pl.smem);
  if (st != RFIM_OK) return st;
  int nclusters = 0;
  if ((st = clusters_per_device_raw(reinterpret_cast<const void*>(kernel), 32 * pl.nw, (size_t)pl.smem, pl.cl, sms,
                                    nclusters)) != RFIM_OK)
    return st;
  if (nclusters < 1) return RFIM_ERR_UNSUPPORTED;
  int64_t want = P.total_tiles;
  if (want > nclusters) want = nclusters;
  if ((st = clear_outputs(c)) != RFIM_OK) return st;
  static const char* names[2][4] = {{"fd_u8_strip1_bulk", "fd_u8_strip2_bulk", "fd_u8_strip4_bulk", "fd_u8_strip8_bulk"},
                                    {"fd_u8_strip1", "fd_u8_strip2", "fd_u8_strip4", "fd_u8_strip8"}};
  static const char* mnames[2] = {"fd_u8_strip1_bulk_median", "fd_u8_strip1_median"};
  return launch(median ? mnames[pl.tensor] : names[pl.tensor][pl.cl == 1 ? 0 : pl.cl == 2 ? 1 : pl.cl == 4 ? 2 : 3], kernel,
                dim3((unsigned)(want * pl.cl)), dim3((unsigned)(32 * pl.nw)), (size_t)pl.smem, c.stream, pl.cl, maps, P);
}

int try_fd_u8_strip(const Call& c, bool want_tensor, int force_cl, int sms) {
  StripPlan sp;
  if (!plan_fd_u8_strip(c, want_tensor, force_cl, sp)) return RFIM_ERR_UNSUPPORTED;
  return launch_fd_strip(c, sp, sms);
}

}  // namespace rfim_host
