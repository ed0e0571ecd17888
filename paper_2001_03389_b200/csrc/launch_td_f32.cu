// launch_td_f32.cu -- geometry and launch of the TDSC float32 kernel (td_f32.cuh).
#include "host.h"
#include "td_f32.cuh"
#include "td_f32_fast.cuh"

namespace rfim_host {

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

// ---- the tuned kernel (td_f32_fast.cuh): whole rows staged in shared memory, windows that are multiples of 4 samples
// (or the whole row), a team of G lanes per window
template <int G>
int launch_td_f32_fast_g(const Call& c, const rfim::TdF32Params& P, int sms, const char* name) {
  const size_t smem = rfim::f32_fast_smem_bytes(P.S, G);
  void (*kernel)(const rfim::TdF32Params) = rfim::td_f32_fast_kernel<G>;
  int st = ensure_smem(kernel, smem);
  if (st != RFIM_OK) return st;
  int occ = 0;
  if ((st = blocks_per_sm(kernel, rfim::kF32FastThreads, smem, occ)) != RFIM_OK) return st;
  if (occ < 1) return RFIM_ERR_UNSUPPORTED;
  int64_t grid = P.rows;
  if (grid > (int64_t)sms * occ) grid = (int64_t)sms * occ;
  if ((st = clear_outputs(c)) != RFIM_OK) return st;
  return launch(name, kernel, dim3((unsigned)grid), dim3(rfim::kF32FastThreads), smem, c.stream, 0, P);
}
int try_td_f32_fast(const Call& c, const rfim::TdF32Params& P, int sms) {
  const uintptr_t a = reinterpret_cast<uintptr_t>(c.data) | reinterpret_cast<uintptr_t>(c.out);
  if ((a & 15) != 0 || (c.stride % 4 != 0 && P.rows != 1) || c.samples % 4 != 0) return RFIM_ERR_UNSUPPORTED;
  const int W = c.window;                               // already clamped to samples
  if (W != c.samples && W % 4 != 0) return RFIM_ERR_UNSUPPORTED;
  if (W > 32768) return RFIM_ERR_UNSUPPORTED;
  const int nwin = (c.samples + W - 1) / W;
  // the smallest team that leaves a lane at most 16 quads (W = 256 -> 4 lanes, 1024 -> 16, 4096 -> 64, longer -> the
  // CTA): short windows keep their scalar chain (square root, bounds, reductions) on few lanes, long ones spread
  int best = 0;
  for (int G = 4; G <= 256; G *= 4) {
    if (W > 64 * G && G != 256) continue;
    if (W > 128 * G) continue;                          // at most 32 quads per lane (bit mask of flagged quads)
    if (rfim::f32_fast_smem_bytes(c.samples, G) > (size_t)kMaxSmem) continue;
    best = G;
    break;
  }
  (void)nwin;
  switch (best) {
    case 4: return launch_td_f32_fast_g<4>(c, P, sms, "td_f32_fast_g4");
    case 16: return launch_td_f32_fast_g<16>(c, P, sms, "td_f32_fast_g16");
    case 64: return launch_td_f32_fast_g<64>(c, P, sms, "td_f32_fast_g64");
    case 256: return launch_td_f32_fast_g<256>(c, P, sms, "td_f32_fast_g256");
    default: return RFIM_ERR_UNSUPPORTED;
  }
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
  // variant 0 / 2: the tuned kernel when the request fits it; 3 / 4: the segment kernel below even then (testing)
  if ((c.variant == 0 || c.variant == 2) && c.reserved_team == 0) {
    st = try_td_f32_fast(c, P, sms);
    if (st != RFIM_ERR_UNSUPPORTED) return st;
  }
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

}  // namespace rfim_host
