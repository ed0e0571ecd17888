// launch_td_u8.cu -- geometry and launch of the TDSC uint8 kernels (td_u8.cuh).
#include "host.h"
#include "td_u8.cuh"

namespace rfim_host {

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

}  // namespace rfim_host
