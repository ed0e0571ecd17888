// td_u8.cuh -- time-domain sigma cut (TDSC, Fig. 2) for uint8 dynamic spectra.
//
// Two kernels:
//   td_u8_staged_kernel   the hot path.  One warp owns one
//       (beam, channel) row at a time.  T1: the row is brought into the warp's shared-memory slot
//       by one 1-D TMA bulk copy (cp.async.bulk, completion on an mbarrier); only the <= 15 head and
//       tail bytes that are not 16-byte aligned in global memory are moved by the lanes.  T2: exact
//       sum and sum of squares with IDP.4A over 16-byte groups.  T3: the cut collapses to two byte
//       bounds, found by evaluating the exact 64/128-bit predicate for all 256 byte values across the
//       warp.  T4: a packed range check (3 instructions per 32-bit word, VIADDMNMX.U16x2) finds the
//       16-byte groups that contain a value outside [lo, hi]; their indices are compacted into a
//       queue and only those groups are revisited byte by byte (replace, update S and Q
//       incrementally).  T5: next threshold, on chip.  T6: one TMA bulk store.  HBM sees one read
//       and one write per sample.
//   td_u8_generic_kernel  any alignment / stride / row length / window, mean or median: one CTA per
//       row, byte loads, iterations through global memory (L1/L2).  Correctness path, not tuned.
#pragma once

#include "common.cuh"

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
  int queue_entries;          // staged kernel: u16 entries per warp queue
};

// ------------------------------------------------------------------------------------------------
// staged hot path
// ------------------------------------------------------------------------------------------------

// Packed range check of one 16-byte group.  For a 32-bit word w, the u16 lanes of w and of w<<8
// carry every byte once as the HIGH byte of a lane, so with LB = lo<<8 a byte lies outside [lo, hi]
// <=> its lane satisfies ((v - LB) mod 2^16) > ((hi-lo)<<8 | 0xFF).  VIADDMNMX.U16x2 does the
// subtract and the running max in one instruction: 3 instructions per word, two chains per group.
__device__ __forceinline__ uint32_t group_range_acc(const uint4& w, uint32_t negLB2) {
  uint32_t a = __viaddmax_u16x2(w.x, negLB2, 0u);
  uint32_t b = __viaddmax_u16x2(w.z, negLB2, 0u);
  a = __viaddmax_u16x2(w.x << 8, negLB2, a);
  b = __viaddmax_u16x2(w.z << 8, negLB2, b);
  a = __viaddmax_u16x2(w.y, negLB2, a);
  b = __viaddmax_u16x2(w.w, negLB2, b);
  a = __viaddmax_u16x2(w.y << 8, negLB2, a);
  b = __viaddmax_u16x2(w.w << 8, negLB2, b);
  return __vmaxu2(a, b);
}

// Append a group index to the warp's hit queue.  Plain shared-memory atomic (inline PTX so that the
// compiler does not wrap it in a ballot/REDUX aggregation): hits are rare, one or two lanes per step.
__device__ __forceinline__ void queue_push(uint32_t tail_addr, uint16_t* queue, int gi) {
  uint32_t at;
  asm volatile("atom.shared.add.u32 %0, [%1], 1;" : "=r"(at) : "r"(tail_addr) : "memory");
  queue[at] = (uint16_t)gi;
}

// Exact mask (0xFF per byte) of the bytes of w outside [lo, hi], 9 instructions: the bytes are spread
// over two words of u16 lanes; lane + (0x7FFF - hi) sets bit 15 iff byte > hi, lane + (0x8000 - lo)
// sets bit 15 iff byte >= lo; PRMT's sign-replicate mode turns the four bit-15 flags into a byte mask.
// chi2 / clo2 hold those constants in both halves.  With lo = 1, hi = 0 every byte is marked.
__device__ __forceinline__ uint32_t prmt(uint32_t a, uint32_t b, uint32_t sel) {
  uint32_t d;
  asm("prmt.b32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(sel));   // selector bit 3 = replicate sign
  return d;
}
__device__ __forceinline__ uint32_t bytes_outside(uint32_t w, uint32_t chi2, uint32_t clo2) {
  const uint32_t xe = prmt(w, 0u, 0x4240u), xo = prmt(w, 0u, 0x4341u);
  const uint32_t fe = (xe + chi2) | ~(xe + clo2);
  const uint32_t fo = (xo + chi2) | ~(xo + clo2);
  return prmt(fe, fo, 0xFBD9u);
}

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

// control block per team (bytes): [0] mbarrier, [8] queue tail, [16] exchange 2 x kTeam(<=2) x 4 u32
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

template <int kTeam, bool kFlags>
__global__ void __launch_bounds__(512 * kTeam, 1) td_u8_staged_kernel(const TdU8Params P) {
  extern __shared__ __align__(128) uint8_t smem[];
  constexpr int TL = 32 * kTeam;                                  // threads per team
  const int lane = threadIdx.x & 31;
  const int team = threadIdx.x / TL;
  const int tl = threadIdx.x % TL;                                // thread index inside the team
  const int wt = tl >> 5;                                         // warp index inside the team
  const int nteams = blockDim.x / TL;
  uint8_t* slot = smem + (size_t)team * P.slot_bytes;
  uint16_t* queue = reinterpret_cast<uint16_t*>(smem + (size_t)nteams * P.slot_bytes) + (size_t)team * P.queue_entries;
  uint8_t* ctrl = smem + (size_t)nteams * P.slot_bytes + (size_t)nteams * P.queue_entries * sizeof(uint16_t) +
                  (size_t)team * kCtrlBytes;
  uint64_t* bar = reinterpret_cast<uint64_t*>(ctrl);
  volatile uint32_t* qtail = reinterpret_cast<volatile uint32_t*>(ctrl + 8);
  volatile uint32_t* xchg = reinterpret_cast<volatile uint32_t*>(ctrl + 16);
  const uint32_t qtail_addr = smem_addr(ctrl + 8);
  if (tl == 0) {
    mbar_init(bar, 1);
    fence_mbar_init();
    *qtail = 0;
  }
  team_sync<kTeam>(team);

  const int S = P.S;
  uint32_t phase = 0;
  int xsel = 0;
  const uint4* s4 = reinterpret_cast<const uint4*>(slot);
  uint32_t* s32 = reinterpret_cast<uint32_t*>(slot);
  const int64_t total_teams = (int64_t)gridDim.x * nteams;
  for (int64_t row = (int64_t)blockIdx.x * nteams + team; row < P.rows; row += total_teams) {
    // ---------------------------------------------------------------- T1: load
    const uint8_t* g = P.src + row * P.stride;
    const RowGeom geo = row_geom(g, S);
    const int h = geo.h, J = geo.J;
    if (tl == 0 && geo.body > 0) {
      mbar_arrive_expect_tx(bar, (uint32_t)geo.body);
      bulk_load(slot + h + geo.a0, g + geo.a0, (uint32_t)geo.body, bar);
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
    if (geo.body > 0) {
      mbar_wait(bar, phase);
      phase ^= 1;
    }
    team_sync<kTeam>(team);

    // ---------------------------------------------------------------- T2: statistics
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
      }
      s1 += s1b; s2 += s2b;
    }
    // totals fit 32 bits: the staged path is limited to S <= 65000 (S*255^2 < 2^32)
    team_sum3<kTeam>(s1, s2, s3, xchg, xsel, wt, lane, team);
    uint32_t xf = slot[h], xl = slot[h + S - 1];
    uint64_t Ssum = s1 - (uint32_t)h * xf - (uint32_t)geo.pe * xl;
    uint64_t Qsum = (uint64_t)s2 - (uint64_t)((uint32_t)h * xf * xf) - (uint64_t)((uint32_t)geo.pe * xl * xl);
    uint32_t qbase = 0;                                           // queue tail only grows within a row

    // ---------------------------------------------------------------- T3..T5: thresholds, on chip
    for (int it = 0; it < P.n_thr; ++it) {
      // T3: exact kept interval [lo, hi] and replacement value for this snapshot (every warp of the
      // team computes the same scalars: cheaper than another barrier)
      int lo, hi;
      const uint64_t V = (uint64_t)S * Qsum - Ssum * Ssum;
      const U8Cut cut = make_cut_u8((uint32_t)S, Ssum, V, P.p[it]);
      warp_bounds_u8_fast(cut, P.pf[it], V, lane, lo, hi);
      if (lo == 0 && hi == 255) continue;                        // nothing can be cut
      const uint32_t r = rounded_mean_u8((uint32_t)S, Ssum);
      const bool all = lo > hi;                                  // empty kept interval: everything is cut
      int qn;
      if (!all) {
        // T4a: packed range check; queue the groups that hold a value outside [lo, hi]
        const uint32_t neg = (0x10000u - ((uint32_t)lo << 8)) & 0xffffu;
        const uint32_t negLB2 = neg | (neg << 16);
        const uint32_t thr = ((uint32_t)(hi - lo) << 8) | 0xffu;
        const uint32_t thr2 = thr | (thr << 16);
        uint16_t* q = queue - qbase;                             // entries of this iteration start at queue[0]
        // four groups per thread in flight (independent loads and compare chains)
        int g0 = 0;
        for (; g0 + 4 * TL <= J; g0 += 4 * TL) {
          const int gi = g0 + tl;
          const uint4 w0 = s4[gi], w1 = s4[gi + TL], w2 = s4[gi + 2 * TL], w3 = s4[gi + 3 * TL];
          const bool h0 = __vmaxu2(group_range_acc(w0, negLB2), thr2) != thr2;
          const bool h1 = __vmaxu2(group_range_acc(w1, negLB2), thr2) != thr2;
          const bool h2 = __vmaxu2(group_range_acc(w2, negLB2), thr2) != thr2;
          const bool h3 = __vmaxu2(group_range_acc(w3, negLB2), thr2) != thr2;
          if (h0) queue_push(qtail_addr, q, gi);
          if (h1) queue_push(qtail_addr, q, gi + TL);
          if (h2) queue_push(qtail_addr, q, gi + 2 * TL);
          if (h3) queue_push(qtail_addr, q, gi + 3 * TL);
        }
        for (; g0 < J; g0 += TL) {
          const int gi = g0 + tl;
          if (gi < J && __vmaxu2(group_range_acc(s4[gi], negLB2), thr2) != thr2) queue_push(qtail_addr, q, gi);
        }
        team_sync<kTeam>(team);
        const uint32_t tail = *qtail;
        qn = (int)(tail - qbase);
        qbase = tail;
      } else {
        for (int gi = tl; gi < J; gi += TL) queue[gi] = (uint16_t)gi;
        qn = J;
        team_sync<kTeam>(team);
      }
      if (qn == 0) continue;
      // T4b: revisit the queued groups, one 32-bit word per thread (8 groups per warp step)
      const uint32_t r4 = r * 0x01010101u;
      const uint32_t chi2 = (0x7fffu - (uint32_t)hi) * 0x00010001u;
      const uint32_t clo2 = (0x8000u - (uint32_t)lo) * 0x00010001u;
      uint32_t cnt = 0, sx = 0, sxx = 0;
      auto fix_word = [&](int widx, uint32_t w) {
        const uint32_t m = bytes_outside(w, chi2, clo2);
        if (m) {
          const uint32_t f = w & m;
          cnt += __popc(m);                                       // 8 per byte; divided below
          sx = __dp4a(f, 0x01010101u, sx);
          sxx = __dp4a(f, f, sxx);
          s32[widx] = (w & ~m) | (r4 & m);
          if (kFlags) {
#pragma unroll
            for (int j = 0; j < 4; ++j) {
              const int i = widx * 4 + j - h;
              if (((m >> (8 * j)) & 1u) && (unsigned)i < (unsigned)S) P.flags[row * S + i] = 1;
            }
          }
        }
      };
      constexpr int EPS = 8 * kTeam;                              // entries per team step
      int e0 = 0;
      for (; e0 + 2 * EPS <= qn; e0 += 2 * EPS) {                 // two independent entries per thread
        const int ea = e0 + (tl >> 2);
        const int wa = (int)queue[ea] * 4 + (tl & 3), wb = (int)queue[ea + EPS] * 4 + (tl & 3);
        const uint32_t va = s32[wa], vb = s32[wb];
        fix_word(wa, va);
        fix_word(wb, vb);
      }
      for (; e0 < qn; e0 += EPS) {
        const int e = e0 + (tl >> 2);
        if (e < qn) {
          const int widx = (int)queue[e] * 4 + (tl & 3);
          fix_word(widx, s32[widx]);
        }
      }
      team_sum3<kTeam>(cnt, sx, sxx, xchg, xsel, wt, lane, team);  // also orders the fixes before the next sweep
      cnt >>= 3;
      if (cnt) {
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
      bulk_store(go + geo.a0, slot + h + geo.a0, (uint32_t)geo.body);
      bulk_commit();
    }
    if (tl < 16) {
      if (tl < geo.a0) go[tl] = slot[h + tl];
    } else if (tl < 32) {
      const int t = tl - 16;
      if (geo.a1 + t < S) go[geo.a1 + t] = slot[h + geo.a1 + t];
    }
    if (tl == 0) {
      if (geo.body > 0) bulk_wait_read<0>();                      // slot may be overwritten after this
      *qtail = 0;
    }
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
