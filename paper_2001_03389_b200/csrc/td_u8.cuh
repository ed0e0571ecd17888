// td_u8.cuh -- time-domain sigma cut (TDSC, Fig. 2) for uint8 dynamic spectra.
//
// Two kernels:
//   td_u8_staged_kernel   the hot path.  One warp owns one
//       (beam, channel) row at a time.  T1: the row is brought into the warp's shared-memory slot
//       by one 1-D TMA bulk copy (cp.async.bulk, completion on an mbarrier); only the <= 15 head and
//       tail bytes that are not 16-byte aligned in global memory are moved by the lanes.  T2: one
//       pass over the row gives the exact sum and sum of squares (IDP.4A) and, per 16-byte group, its
//       largest and smallest byte (VIMNMX3.U16x2) -- the group summaries.  T3: the cut collapses to
//       two byte bounds, found by evaluating the exact 64/128-bit predicate on candidate byte values
//       across the warp.  T4: a threshold sweep reads only the summaries (two bytes per group instead
//       of sixteen): a packed test per sixteen groups, exact byte masks where it fires; a lane repairs
//       the groups it found by itself (exact per-byte masks, replace, S and Q deltas, summary
//       refresh), so there is no queue, atomic or barrier.  T5: next threshold, on chip, from the
//       updated S, Q and summaries.  T6: one TMA bulk store.  HBM sees one read and one write per
//       sample.  Median replacement (kMedian): the replacement value is the lower median of the
//       snapshot, found -- only in rows where an iteration cuts something, at the first hit and therefore before
//       any replacement -- by counting passes over the staged row (bytes <= v, packed compares + IDP.4A) that start
//       at the rounded mean and bracket, then bisect, the rank; it is the same for every later iteration.
//   td_u8_generic_kernel  any alignment / stride / row length / window, mean or median: one CTA per
//       row, byte loads, iterations through global memory (L1/L2).  Correctness path, not tuned.
#pragma once

#include "common.cuh"
#include "packed.cuh"

namespace rfim {

struct TdU8Params {
  const uint8_t* src;
  uint8_t* dst;
  int64_t rows;
  int64_t stride;
  int S;
  int window;                 // generic kernel only; >= 1
  int n_thr;
  int policy;                 // generic kernel only
  uint32_t p[16];             // thresholds as p / 2^16
  float pf[16];               // the same thresholds as floats (estimates only)
  uint8_t* flags;             // optional [rows][S]
  unsigned long long* counts; // optional [n_thr]
  int slot_bytes;             // staged kernel: bytes per warp slot (multiple of 16)
  int sum_entries;            // staged kernel: group summaries per team (a multiple of 16)
};

// ------------------------------------------------------------------------------------------------
// staged hot path
// ------------------------------------------------------------------------------------------------

// Kept interval [lo, hi] for one cut, fast form: a float estimate of mu -/+ k sigma picks 16
// candidate values per side; the EXACT integer predicate is evaluated on them (one per lane) and the
// transition is read off with two ballots.  If a window does not contain its transition (estimate
// off, empty interval) the full 256-value scan decides.  Result identical to warp_bounds_u8.
__device__ __forceinline__ void warp_bounds_u8_fast(const U8Cut& c, float k, uint64_t V, int lane,
                                                    int& lo, int& hi) {
  const float rn = __frcp_rn((float)c.N);
  const float mu = (float)c.S * rn;
  const float vf = (float)V;
  const float ks = k * (vf * rsqrtf(fmaxf(vf, 1.0f))) * rn;      // only an estimate: the exact test decides
  const int glo = (int)fminf(fmaxf(ceilf(mu - ks), 0.0f), 255.0f);
  const int ghi = (int)fminf(fmaxf(floorf(mu + ks), 0.0f), 255.0f);
  const bool low_side = lane < 16;
  const int x = low_side ? glo - 8 + lane : ghi - 7 + (lane - 16);
  const bool inside = x >= 0 && x <= 255;
  const bool kept = inside && !cut_flags_u8(c, (uint32_t)x);
  // values outside 0..255 count as "cut" sentinels on both ends
  const uint32_t kb = __ballot_sync(FULL, kept);
  const uint32_t klo = kb & 0xffffu, khi = kb >> 16;
  bool ok = klo != 0 && khi != 0;
  if (ok) {
    const int f = __ffs(klo) - 1;                // first kept candidate on the low side
    const int l = 31 - __clz(khi);               // last kept candidate on the high side (0..15)
    // The kept set is an interval, so the first kept candidate is its lower end provided the
    // candidate below it exists in the window (it is then cut) or is -1; same at the upper end.
    lo = glo - 8 + f;
    hi = ghi - 7 + l;
    if (f == 0 && lo > 0) ok = false;
    if (l == 15 && hi < 255) ok = false;
  }
  if (!ok) warp_bounds_u8(c, lane, lo, hi);
}

// T2m: number of bytes <= v among the J 16-byte groups of a staged row (padding included), by one warp
__device__ __forceinline__ uint32_t warp_count_le(const uint4* s4, int J, uint32_t v, int lane) {
  const uint32_t cab2 = (0x7fffu - v) * 0x00010001u;              // bytes_above(w, cab2): bytes > v
  uint32_t n = 0;
  for (int gi = lane; gi < J; gi += 32) {
    const uint4 w = s4[gi];
    n = __dp4a(~bytes_above(w.x, cab2) & 0x01010101u, 0x01010101u, n);
    n = __dp4a(~bytes_above(w.y, cab2) & 0x01010101u, 0x01010101u, n);
    n = __dp4a(~bytes_above(w.z, cab2) & 0x01010101u, 0x01010101u, n);
    n = __dp4a(~bytes_above(w.w, cab2) & 0x01010101u, 0x01010101u, n);
  }
  return __reduce_add_sync(FULL, n);
}
// Lower median (rank (S - 1) / 2 of the ascending snapshot) of the row staged at slot[h .. h + S): the smallest v
// with #{x <= v} > rank.  hpad / epad copies of xf / xl pad the first / last group and are taken out of every
// count.  The search starts at `guess` (the rounded mean), gallops to a bracket and bisects: two or three
// counting passes for noise-like rows, at most about twelve.
__device__ __forceinline__ uint32_t warp_lower_median_u8(const uint4* s4, int J, int S, int hpad, int epad, uint32_t xf,
                                                         uint32_t xl, uint32_t guess, int lane) {
  const uint32_t rank = (uint32_t)(S - 1) >> 1;
  auto above = [&](uint32_t v) {                                  // #{x <= v} > rank ?
    uint32_t n = warp_count_le(s4, J, v, lane);
    n -= (xf <= v ? (uint32_t)hpad : 0u) + (xl <= v ? (uint32_t)epad : 0u);
    return n > rank;
  };
  int lo, hi;                                                     // the median lies in [lo, hi]
  int g = (int)min(guess, 255u);
  if (above((uint32_t)g)) {
    hi = g; lo = 0;
    for (int step = 1; hi - step >= 0; step <<= 1) {
      if (above((uint32_t)(hi - step))) { hi -= step; } else { lo = hi - step + 1; break; }
    }
  } else {
    lo = g + 1; hi = 255;
    for (int step = 1; lo + step - 1 <= 255; step <<= 1) {
      if (above((uint32_t)(lo + step - 1))) { hi = lo + step - 1; break; } else { lo += step; }
    }
  }
  while (lo < hi) {
    const int mid = (lo + hi) >> 1;
    if (above((uint32_t)mid)) hi = mid; else lo = mid + 1;
  }
  return (uint32_t)lo;
}

// A team of kTeam warps (1 or 2) owns one shared-memory slot and one row at a time; sixteen teams
// per SM keep sixteen rows in flight, which is what covers the HBM latency (measured: fewer teams
// with two slots each are slower).  kTeam = 2 doubles the warps per SM for the same shared memory.
template <int kTeam>
__device__ __forceinline__ void team_sync(int team) {
  if (kTeam == 1) __syncwarp();
  else asm volatile("bar.sync %0, %1;" ::"r"(team), "n"(32 * kTeam) : "memory");
}

// sum three lane values over the team: warp REDUX, then partials exchanged through shared memory
template <int kTeam>
__device__ __forceinline__ void team_sum3(uint32_t& a, uint32_t& b, uint32_t& c, volatile uint32_t* xchg,
                                          int& xsel, int wt, int lane, int team) {
  a = __reduce_add_sync(FULL, a);
  b = __reduce_add_sync(FULL, b);
  c = __reduce_add_sync(FULL, c);
  if (kTeam == 1) { __syncwarp(); return; }
  volatile uint32_t* buf = xchg + xsel * (kTeam * 4);      // double-buffered: one barrier per exchange
  if (lane == 0) { buf[wt * 4 + 0] = a; buf[wt * 4 + 1] = b; buf[wt * 4 + 2] = c; }
  team_sync<kTeam>(team);
  a = 0; b = 0; c = 0;
#pragma unroll
  for (int w = 0; w < kTeam; ++w) { a += buf[w * 4 + 0]; b += buf[w * 4 + 1]; c += buf[w * 4 + 2]; }
  xsel ^= 1;
}

// control block per team (bytes): [0] mbarrier, [16] exchange 2 x kTeam(<=2) x 4 u32
constexpr int kCtrlBytes = 16 + 2 * 2 * 4 * 4;

// geometry of one row inside its slot: row byte i lives at slot[h + i]
struct RowGeom {
  int h;      // misalignment of the row start in global memory (0..15)
  int a0;     // bytes before the first 16-byte aligned global address (head, moved by lanes)
  int body;   // aligned interior moved by TMA (multiple of 16)
  int a1;     // a0 + body: first tail byte
  int J;      // 16-byte groups covering [0, h + S)
  int pe;     // padding bytes behind the row
};
__device__ __forceinline__ RowGeom row_geom(const uint8_t* g, int S) {
  RowGeom r;
  r.h = (int)(reinterpret_cast<uintptr_t>(g) & 15);
  r.a0 = (16 - r.h) & 15;
  if (r.a0 > S) r.a0 = S;
  r.body = (S - r.a0) & ~15;
  r.a1 = r.a0 + r.body;
  r.J = (r.h + S + 15) >> 4;
  r.pe = 16 * r.J - (r.h + S);
  return r;
}

template <int kTeam, bool kFlags, bool kMedian>
__global__ void __launch_bounds__(512 * kTeam, 1) td_u8_staged_kernel(const TdU8Params P) {
  static_assert(!(kMedian && kTeam != 1), "the snapshot median is taken by the one warp that owns the row");
  extern __shared__ __align__(128) uint8_t smem[];
  constexpr int TL = 32 * kTeam;                                  // threads per team
  const int lane = threadIdx.x & 31;
  const int team = threadIdx.x / TL;
  const int tl = threadIdx.x % TL;                                // thread index inside the team
  const int wt = tl >> 5;                                         // warp index inside the team
  const int nteams = blockDim.x / TL;
  // shared memory: [slots][group summaries][control blocks], one of each per team
  uint8_t* slot = smem + (size_t)team * P.slot_bytes;
  uint8_t* base = smem + (size_t)nteams * P.slot_bytes;
  uint8_t* gmax = base + (size_t)team * P.sum_entries * 2;        // largest byte of every 16-byte group
  uint8_t* gmin = gmax + P.sum_entries;                           // smallest byte
  base += (size_t)nteams * P.sum_entries * 2;
  uint8_t* ctrl = base + (size_t)team * kCtrlBytes;
  uint64_t* bar = reinterpret_cast<uint64_t*>(ctrl);
  volatile uint32_t* xchg = reinterpret_cast<volatile uint32_t*>(ctrl + 16);
  if (tl == 0) {
    mbar_init(bar, 1);
    fence_mbar_init();
  }
  team_sync<kTeam>(team);

  const int S = P.S;
  uint32_t phase = 0;
  int xsel = 0;
  // A row is read once and written once: both copies carry L2 evict-first, so that what stays in L2 is what is still
  // needed -- the rows the teams have PREFETCHED (normal priority).  Without the hints the 9.2 GB of stores pushed
  // prefetched lines out before their copy-in arrived: 10.27 GB of DRAM reads for a 9.22 GB batch; with them 9.30 GB
  // and 1.3 % less time (profiles/r2k_td_u8_hints.md).
  const uint64_t stream_once = l2_policy_evict_first();
  const uint4* s4 = reinterpret_cast<const uint4*>(slot);
  const uint4* gmax4 = reinterpret_cast<const uint4*>(gmax);
  const uint4* gmin4 = reinterpret_cast<const uint4*>(gmin);
  const int64_t total_teams = (int64_t)gridDim.x * nteams;
  for (int64_t row = (int64_t)blockIdx.x * nteams + team; row < P.rows; row += total_teams) {
    // ---------------------------------------------------------------- T1: load
    const uint8_t* g = P.src + row * P.stride;
    const RowGeom geo = row_geom(g, S);
    const int h = geo.h, J = geo.J;
    if (tl == 0 && geo.body > 0) {
      mbar_arrive_expect_tx(bar, (uint32_t)geo.body);
      bulk_load_hint(slot + h + geo.a0, g + geo.a0, (uint32_t)geo.body, bar, stream_once);
    }
    // Padding is filled with COPIES of the first / last sample: the decision depends only on the
    // value, so the copies always share their original's fate and are subtracted again below.
    if (tl < 16) {
      if (tl < h) slot[tl] = g[0];
      if (tl < geo.a0) slot[h + tl] = g[tl];                     // head bytes
    } else if (tl < 32) {
      const int t = tl - 16;
      if (geo.a1 + t < S) slot[h + geo.a1 + t] = g[geo.a1 + t];  // tail bytes
      if (t < geo.pe) slot[h + S + t] = g[S - 1];
    }
    const int J16 = (J + 15) >> 4;                                // summaries are swept sixteen at a time
    if (tl < 16 && J + tl < 16 * J16) { gmax[J + tl] = 0; gmin[J + tl] = 255; }   // neutral: no cut touches them
    if (geo.body > 0) {
      mbar_wait(bar, phase);
      phase ^= 1;
    }
    team_sync<kTeam>(team);

    // ---------------------------------------------------------------- T2: statistics and group summaries
    uint32_t s1 = 0, s2 = 0, s3 = 0;
    {
      uint32_t s1b = 0, s2b = 0;
#pragma unroll 4
      for (int gi = tl; gi < J; gi += TL) {
        const uint4 w = s4[gi];
        s1 = __dp4a(w.x, 0x01010101u, s1); s2 = __dp4a(w.x, w.x, s2);
        s1b = __dp4a(w.y, 0x01010101u, s1b); s2b = __dp4a(w.y, w.y, s2b);
        s1 = __dp4a(w.z, 0x01010101u, s1); s2 = __dp4a(w.z, w.z, s2);
        s1b = __dp4a(w.w, 0x01010101u, s1b); s2b = __dp4a(w.w, w.w, s2b);
        const uint32_t e = group_summary(w);
        gmax[gi] = (uint8_t)(e >> 8);
        gmin[gi] = (uint8_t)e;
      }
      s1 += s1b; s2 += s2b;
    }
    // the team's next row travels HBM -> L2 while this one is iterated; its copy then comes from L2
    if (tl == 0 && row + total_teams < P.rows) {
      const uint8_t* gn = g + total_teams * P.stride;
      const RowGeom gnx = row_geom(gn, S);
      if (gnx.body > 0) bulk_prefetch_l2(gn + gnx.a0, (uint32_t)gnx.body);
    }
    // totals fit 32 bits: the staged path is limited to S <= 65000 (S*255^2 < 2^32)
    team_sum3<kTeam>(s1, s2, s3, xchg, xsel, wt, lane, team);
    uint32_t xf = slot[h], xl = slot[h + S - 1];
    uint64_t Ssum = s1 - (uint32_t)h * xf - (uint32_t)geo.pe * xl;
    uint64_t Qsum = (uint64_t)s2 - (uint64_t)((uint32_t)h * xf * xf) - (uint64_t)((uint32_t)geo.pe * xl * xl);

    // ---------------------------------------------------------------- T3..T5: thresholds, on chip
    uint4* s4w = reinterpret_cast<uint4*>(slot);
    bool have_med = false;                                         // kMedian: the row's lower median, once known
    uint32_t med = 0;
    for (int it = 0; it < P.n_thr; ++it) {
      // T3: exact kept interval [lo, hi] for this snapshot (every warp of the team computes the same
      // scalars: cheaper than another barrier)
      int lo, hi;
      const uint64_t V = (uint64_t)S * Qsum - Ssum * Ssum;
      const U8Cut cut = make_cut_u8((uint32_t)S, Ssum, V, P.p[it]);
      warp_bounds_u8_fast(cut, P.pf[it], V, lane, lo, hi);
      if (lo == 0 && hi == 255) continue;                        // nothing can be cut
      const bool upd = it + 1 < P.n_thr;                         // later sweeps need fresh summaries
      const uint32_t HI2 = (((uint32_t)(hi & 0xff) << 8) | 0xffu) * 0x00010001u;
      const uint32_t LO2 = ((uint32_t)lo << 8) * 0x00010001u;
      const uint32_t cab2 = (0x7fffu - (uint32_t)(hi & 0xff)) * 0x00010001u;
      const uint32_t cbe2 = (0x7fffu + (uint32_t)lo) * 0x00010001u;
      const uint32_t chi2 = (0x7fffu - (uint32_t)hi) * 0x00010001u;
      const uint32_t clo2 = (0x8000u - (uint32_t)lo) * 0x00010001u;
      uint32_t r = 0, r4 = 0;
      bool have_r = false;
      uint32_t cnt = 0, sx = 0, sxx = 0;
      // T4b: a lane repairs a whole 16-byte group by itself: exact byte masks, replace, accumulate the
      // deltas of S and Q, refresh the group's summary.  Groups are private to the lane that swept their
      // summaries, so no queue, atomic or barrier is involved.
      auto fix_word = [&](uint32_t w, int widx) -> uint32_t {   // branch-free: most lanes see m == 0
        const uint32_t m = bytes_outside(w, chi2, clo2);
        const uint32_t f = w & m;
        cnt += __popc(m);                                         // 8 per byte; divided below
        sx = __dp4a(f, 0x01010101u, sx);
        sxx = __dp4a(f, f, sxx);
        if (kFlags && m) {
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            const int i = widx * 4 + j - h;
            if (((m >> (8 * j)) & 1u) && (unsigned)i < (unsigned)S) P.flags[row * S + i] = 1;
          }
        }
        return (w & ~m) | (r4 & m);
      };
      // T4a: sweep the group summaries, sixteen groups per lane and step
      for (int ub = 0; ub < J16; ub += TL) {
        const int u = ub + tl;
        uint4 a = make_uint4(0u, 0u, 0u, 0u), b = make_uint4(~0u, ~0u, ~0u, ~0u);
        if (u < J16) { a = gmax4[u]; b = gmin4[u]; }
        uint32_t ah = __vimax3_u16x2(a.x, a.y, a.z), al = __vimin3_u16x2(b.x, b.y, b.z);
        ah = __vimax3_u16x2(ah, a.w, a.x << 8);      al = __vimin3_u16x2(al, b.w, b.x << 8);
        ah = __vimax3_u16x2(ah, a.y << 8, a.z << 8); al = __vimin3_u16x2(al, b.y << 8, b.z << 8);
        ah = __vimax3_u16x2(ah, a.w << 8, HI2);      al = __vimin3_u16x2(al, b.w << 8, LO2);
        const bool hit = ah != HI2 || al != LO2;
        if (!__any_sync(FULL, hit)) continue;
        if (!have_r) {
          // first hit of this iteration: nothing has been replaced yet, the slot still holds the snapshot
          r = rounded_mean_u8((uint32_t)S, Ssum);
          if (kMedian) {
            // The lower median is taken ONCE per row: replacing samples by the lower median m never changes it (with
            // L samples < m and E samples = m, L <= rank < L + E; moving l samples from below and u from above onto
            // m leaves L - l <= rank < L + E + u), so every later iteration's snapshot median is the same m.
            if (!have_med) { med = warp_lower_median_u8(s4, J, S, h, geo.pe, xf, xl, r, lane); have_med = true; }
            r = med;
          }
          r4 = r * 0x01010101u;
          have_r = true;
        }
        if (hit) {
          // exact hit mask: bit j <=> group 16 u + j holds a value outside [lo, hi]
          const uint32_t m0 = bytes_above(a.x, cab2) | bytes_below(b.x, cbe2);
          const uint32_t m1 = bytes_above(a.y, cab2) | bytes_below(b.y, cbe2);
          const uint32_t m2 = bytes_above(a.z, cab2) | bytes_below(b.z, cbe2);
          const uint32_t m3 = bytes_above(a.w, cab2) | bytes_below(b.w, cbe2);
          uint32_t hm = (((m0 & 0x01010101u) * 0x01020408u) >> 24) | ((((m1 & 0x01010101u) * 0x01020408u) >> 24) << 4) |
                        ((((m2 & 0x01010101u) * 0x01020408u) >> 24) << 8) | ((((m3 & 0x01010101u) * 0x01020408u) >> 24) << 12);
          while (hm) {
            const int gi = u * 16 + __ffs(hm) - 1;
            hm &= hm - 1;
            uint4 w = s4w[gi];
            w.x = fix_word(w.x, gi * 4 + 0);
            w.y = fix_word(w.y, gi * 4 + 1);
            w.z = fix_word(w.z, gi * 4 + 2);
            w.w = fix_word(w.w, gi * 4 + 3);
            s4w[gi] = w;
            if (upd) {
              const uint32_t e = group_summary(w);
              gmax[gi] = (uint8_t)(e >> 8);
              gmin[gi] = (uint8_t)e;
            }
          }
        }
      }
      if (kTeam == 1 && !have_r) continue;                          // no group was touched (have_r is warp-uniform)
      team_sum3<kTeam>(cnt, sx, sxx, xchg, xsel, wt, lane, team);  // also orders the fixes before the next sweep
      cnt >>= 3;
      if (cnt) {
        if (!have_r) r = rounded_mean_u8((uint32_t)S, Ssum);     // the hits were in another warp of the team
        // take the padding copies out again: they were cut iff their original was
        const bool ff = (int)xf < lo || (int)xf > hi, fl = (int)xl < lo || (int)xl > hi;
        if (ff) { cnt -= h; sx -= h * xf; sxx -= h * xf * xf; xf = r; }
        if (fl) { cnt -= geo.pe; sx -= geo.pe * xl; sxx -= geo.pe * xl * xl; xl = r; }
        Ssum = Ssum + (uint64_t)cnt * r - sx;
        Qsum = Qsum + (uint64_t)cnt * r * r - sxx;
        if (tl == 0 && P.counts && cnt) atomicAdd(&P.counts[it], (unsigned long long)cnt);
      }
    }

    // ---------------------------------------------------------------- T6: store
    uint8_t* go = P.dst + row * P.stride;
    fence_proxy_async_smem();
    team_sync<kTeam>(team);
    if (tl == 0 && geo.body > 0) {
      bulk_store_hint(go + geo.a0, slot + h + geo.a0, (uint32_t)geo.body, stream_once);
      bulk_commit();
    }
    if (tl < 16) {
      if (tl < geo.a0) go[tl] = slot[h + tl];
    } else if (tl < 32) {
      const int t = tl - 16;
      if (geo.a1 + t < S) go[geo.a1 + t] = slot[h + geo.a1 + t];
    }
    if (tl == 0 && geo.body > 0) bulk_wait_read<0>();             // slot may be overwritten after this
    team_sync<kTeam>(team);
  }
}

// ------------------------------------------------------------------------------------------------
// generic path
// ------------------------------------------------------------------------------------------------
constexpr int kGenericThreads = 256;

__device__ __forceinline__ uint64_t block_sum_u64(uint64_t v, uint64_t* red) {
  v = warp_sum_u64(v);
  __syncthreads();
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
  __syncthreads();
  uint64_t t = 0;
  for (int w = 0; w < (int)(blockDim.x >> 5); ++w) t += red[w];
  return t;
}

// lower median (rank (n-1)/2) from a 256-bin histogram, computed by warp 0; result to *out
__device__ __forceinline__ void warp_hist_median(const uint32_t* hist, uint32_t n, int lane, int* out) {
  uint32_t c[8], tot = 0;
#pragma unroll
  for (int j = 0; j < 8; ++j) { c[j] = hist[lane * 8 + j]; tot += c[j]; }
  uint32_t incl = tot;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const uint32_t t = __shfl_up_sync(FULL, incl, o);
    if (lane >= o) incl += t;
  }
  const uint32_t rank = (n - 1) / 2;
  uint32_t before = incl - tot;                                   // values in lower lanes
  if (rank >= before && rank < incl) {
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      if (rank < before + c[j]) { *out = lane * 8 + j; break; }
      before += c[j];
    }
  }
}

__global__ void __launch_bounds__(kGenericThreads) td_u8_generic_kernel(const TdU8Params P) {
  __shared__ uint64_t red[kGenericThreads / 32];
  __shared__ uint32_t hist[256];
  __shared__ int sh_lo, sh_hi, sh_r;
  const int tid = threadIdx.x, lane = tid & 31;
  for (int64_t row = blockIdx.x; row < P.rows; row += gridDim.x) {
    const uint8_t* s = P.src + row * P.stride;
    uint8_t* d = P.dst + row * P.stride;
    for (int w0 = 0; w0 < P.S; w0 += P.window) {
      const int n = min(P.window, P.S - w0);
      uint64_t a = 0, b = 0;
      for (int i = tid; i < n; i += kGenericThreads) {
        const uint32_t x = s[w0 + i];
        if (d != s) d[w0 + i] = (uint8_t)x;
        a += x; b += x * x;
      }
      uint64_t Ssum = block_sum_u64(a, red);
      uint64_t Qsum = block_sum_u64(b, red);
      for (int it = 0; it < P.n_thr; ++it) {
        if (P.policy == 1) {                                      // lower median of the snapshot
          for (int i = tid; i < 256; i += kGenericThreads) hist[i] = 0;
          __syncthreads();
          for (int i = tid; i < n; i += kGenericThreads) atomicAdd(&hist[d[w0 + i]], 1u);
          __syncthreads();
        }
        if (tid < 32) {
          const U8Cut cut = make_cut_u8((uint32_t)n, Ssum, (uint64_t)n * Qsum - Ssum * Ssum, P.p[it]);
          int lo, hi;
          warp_bounds_u8(cut, lane, lo, hi);
          if (lane == 0) { sh_lo = lo; sh_hi = hi; }
          if (P.policy == 1) warp_hist_median(hist, (uint32_t)n, lane, &sh_r);
          else if (lane == 0) sh_r = (int)rounded_mean_u8((uint32_t)n, Ssum);
        }
        __syncthreads();
        const int lo = sh_lo, hi = sh_hi;
        const uint32_t r = (uint32_t)sh_r;
        uint64_t cnt = 0, sx = 0, sxx = 0;
        if (!(lo == 0 && hi == 255)) {
          for (int i = tid; i < n; i += kGenericThreads) {
            const uint32_t x = d[w0 + i];
            if ((int)x < lo || (int)x > hi) {
              d[w0 + i] = (uint8_t)r;
              ++cnt; sx += x; sxx += x * x;
              if (P.flags) P.flags[row * P.S + w0 + i] = 1;
            }
          }
        }
        cnt = block_sum_u64(cnt, red);
        sx = block_sum_u64(sx, red);
        sxx = block_sum_u64(sxx, red);
        Ssum = Ssum + cnt * r - sx;
        Qsum = Qsum + cnt * r * r - sxx;
        if (tid == 0 && P.counts && cnt) atomicAdd(&P.counts[it], (unsigned long long)cnt);
        __syncthreads();
      }
    }
  }
}

}  // namespace rfim
