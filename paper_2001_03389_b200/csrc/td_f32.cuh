// td_f32.cuh -- time-domain sigma cut (TDSC, Fig. 2) for float32 dynamic spectra, with
// statistics windows and mean / lower-median replacement (BASELINE.json configs[4]).
//
// One kernel, td_f32_kernel<kTW, kStage>:
//   A CTA of 256 threads owns one SEGMENT at a time: a run of whole statistics windows of one
//   (beam, channel) row (the whole row when it fits: 12500 float32 = 50 KB).  T1: the segment is
//   brought into shared memory by one 1-D TMA bulk copy (rows of float32 are 16-byte aligned whenever
//   the pitch is a multiple of 4; otherwise by coalesced loads).  The CTA's warps form TEAMS of kTW
//   warps; a team owns one window at a time.
//   T2: one pass, fp64: A = sum (x - c), B = sum (x - c)^2 around the pivot c = x[0] of the window
//       (mu = c + A/N, sigma^2 = B/N - (A/N)^2); when the pivot turns out to be far from the mean in units
//       of sigma (a spike at x[0], or after a huge sample was replaced) the sums are taken again around
//       the mean, so the subtraction never loses more than six digits.
//   T3: cut = k sigma in fp64; the fp64 test |x - mu| > cut is monotone in x on each side, so it
//       equals two float compares x > t_hi, x < t_lo, with t_hi / t_lo found by evaluating the fp64
//       predicate on the floats next to fl(mu +- cut).  The sweep is therefore exactly the fp64 test.
//   T2m: lower median (rank (N-1)/2) only in windows that flag something: monotone 258-bin
//       histogram of the window guided by mu and sigma, the bin that holds the rank is compacted and
//       ranked; bins that are too full are split again (generic refinement), with a key-space
//       bisection as the guaranteed-to-finish last resort.
//   T4: flagged samples are replaced; A and B are updated with the fp64 deltas of the replaced
//       samples only.  T5: next threshold on chip.  T6: one TMA bulk store.
//   kStage = false: same code working in place on global memory (any window / row length).
#pragma once

#include "common.cuh"

namespace rfim {

struct TdF32Params {
  const float* src;
  float* dst;
  int64_t rows;
  int64_t stride;
  int S;
  int window;
  int n_thr;
  int policy;
  double k[16];
  uint8_t* flags;               // optional [rows][S]
  unsigned long long* counts;   // optional [n_thr]
  int seg;                      // samples per segment (a multiple of window, or S)
  int segs_per_row;
  int bulk;                     // 1: segments are 16-byte aligned in src and dst -> TMA bulk copies
};

constexpr int kF32Threads = 256;
constexpr int kF32HistBins = 288;     // 258 used (open-ended bin 0, 256 inner bins, open-ended bin 257), padded to 32 * 9
constexpr int kF32ListCap = 64;

// per-team scratch in shared memory
struct __align__(16) F32Team {
  uint32_t hist[kF32HistBins];
  float list[kF32ListCap];
  double red[2][8][2];            // double-buffered exchange of two doubles per warp of the team
  uint32_t redu[2][8][2];
  int ln;                         // compaction cursor
  int beta, below, m;             // bin that holds the rank, elements below it, elements in it
  float result;
  int xsel;
};

template <int kTW>
__device__ __forceinline__ void f32_team_sync(int team) {
  if (kTW == 1) __syncwarp();
  else if (kTW == kF32Threads / 32) __syncthreads();
  else asm volatile("bar.sync %0, %1;" ::"r"(team + 1), "n"(32 * kTW) : "memory");
}

// sum of two doubles over the team (result in every thread); `sel` alternates the exchange buffer so
// that one barrier per reduction is enough
template <int kTW>
__device__ __forceinline__ void f32_team_sum2(double& a, double& b, F32Team* T, int& sel, int wt, int lane, int team) {
  a = warp_sum_f64(a);
  b = warp_sum_f64(b);
  if (kTW == 1) return;
  if (lane == 0) { T->red[sel][wt][0] = a; T->red[sel][wt][1] = b; }
  f32_team_sync<kTW>(team);
  a = 0.0; b = 0.0;
#pragma unroll
  for (int w = 0; w < kTW; ++w) { a += T->red[sel][w][0]; b += T->red[sel][w][1]; }
  sel ^= 1;
}
template <int kTW>
__device__ __forceinline__ uint32_t f32_team_sum_u32(uint32_t a, F32Team* T, int& sel, int wt, int lane, int team) {
  a = __reduce_add_sync(FULL, a);
  if (kTW == 1) return a;
  if (lane == 0) T->redu[sel][wt][0] = a;
  f32_team_sync<kTW>(team);
  a = 0;
#pragma unroll
  for (int w = 0; w < kTW; ++w) a += T->redu[sel][w][0];
  sel ^= 1;
  return a;
}

__device__ __forceinline__ float f32_next_up(float x) {
  if (x == 0.0f) return __int_as_float(1);
  const int b = __float_as_int(x);
  return __int_as_float(x > 0.0f ? b + 1 : b - 1);
}
__device__ __forceinline__ float f32_next_down(float x) {
  if (x == 0.0f) return __int_as_float((int)0x80000001u);
  const int b = __float_as_int(x);
  return __int_as_float(x > 0.0f ? b - 1 : b + 1);
}

// T3: float bounds equivalent to the fp64 test.  flag <=> fabs((double)x - mu) > cut
//   <=> ((double)x - mu) > cut  or  (mu - (double)x) > cut;  both sides are monotone in x, so
//   flag <=> x > t_hi or x < t_lo with t_hi the largest float that the first test keeps and t_lo the
//   smallest float that the second test keeps.
__device__ __forceinline__ void f32_bounds(double mu, double cut, float& t_lo, float& t_hi) {
  const float inf = __int_as_float(0x7f800000);
  float h = __double2float_rd(mu + cut);
  if (h == inf) h = 3.402823466e38f;
  while (h > -3.402823466e38f && ((double)h - mu) > cut) h = f32_next_down(h);
  while (h < 3.402823466e38f && !(((double)f32_next_up(h) - mu) > cut)) h = f32_next_up(h);
  float l = __double2float_ru(mu - cut);
  if (l == -inf) l = -3.402823466e38f;
  while (l < 3.402823466e38f && (mu - (double)l) > cut) l = f32_next_up(l);
  while (l > -3.402823466e38f && !((mu - (double)f32_next_down(l)) > cut)) l = f32_next_down(l);
  t_lo = l;
  t_hi = h;
}

// order-preserving key of a float (for the bisection of last resort); -0 and +0 get the same key
__device__ __forceinline__ uint32_t f32_key(float x) {
  const uint32_t b = (x == 0.0f) ? 0u : (uint32_t)__float_as_int(x);
  return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}

// monotone (non-decreasing) map of a value to one of 258 bins
__device__ __forceinline__ int f32_bin(float x, float vlo, float scale) {
  const int b = __float2int_rd((x - vlo) * scale);
  return min(max(b, -1), 256) + 1;
}

// ------------------------------------------------------------------------------------------------
// T2m: lower median of the n values x[0..n) by the whole team.  Every thread returns the value.
// The values are only read.  mu / sigma (floats, estimates) guide the first histogram.
// ------------------------------------------------------------------------------------------------
template <int kTW>
__device__ float f32_team_median(const float* x, int n, float muf, float sigf, F32Team* T, int tl, int lane,
                                 int team) {
  constexpr int TT = 32 * kTW;
  const int rho = (n - 1) >> 1;
  // guided level: 256 inner bins over mu +- 10 sigma / sqrt(n) (the median of n Gaussian draws is
  // within 1.25 sigma / sqrt(n) of the mean at one standard deviation)
  float R = 10.0f * sigf * rsqrtf((float)n);
  float vlo = muf - R;
  float scale = 128.0f / R;
  if (!(scale < 1e30f)) scale = 1e30f;
  for (int level = 0; level < 48; ++level) {
    for (int i = tl; i < kF32HistBins; i += TT) T->hist[i] = 0;
    if (tl == 0) T->ln = 0;
    f32_team_sync<kTW>(team);
#pragma unroll 4
    for (int i = tl; i < n; i += TT) atomicAdd(&T->hist[f32_bin(x[i], vlo, scale)], 1u);
    f32_team_sync<kTW>(team);
    if (tl < 32) {                                       // leader warp: the bin that holds rank rho
      uint32_t c[9], tot = 0;
#pragma unroll
      for (int j = 0; j < 9; ++j) { c[j] = T->hist[lane * 9 + j]; tot += c[j]; }
      uint32_t incl = tot;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const uint32_t t = __shfl_up_sync(FULL, incl, o);
        if (lane >= o) incl += t;
      }
      uint32_t before = incl - tot;
      if ((uint32_t)rho >= before && (uint32_t)rho < incl) {
#pragma unroll
        for (int j = 0; j < 9; ++j) {
          if ((uint32_t)rho < before + c[j]) { T->beta = lane * 9 + j; T->below = (int)before; T->m = (int)c[j]; break; }
          before += c[j];
        }
      }
    }
    f32_team_sync<kTW>(team);
    const int beta = T->beta, m = T->m, t = rho - T->below;
    if (m <= kF32ListCap) {
      // compact the bin and rank its elements
      for (int i = tl; i < n; i += TT) {
        const float v = x[i];
        if (f32_bin(v, vlo, scale) == beta) T->list[atomicAdd(&T->ln, 1)] = v;
      }
      f32_team_sync<kTW>(team);
      if (tl < 32) {
        for (int i = lane; i < m; i += 32) {
          const float e = T->list[i];
          int rank = 0;
          for (int j = 0; j < m; ++j) {
            const float o = T->list[j];
            rank += (o < e) || (o == e && j < i);
          }
          if (rank == t) T->result = e;
        }
      }
      f32_team_sync<kTW>(team);
      const float r = T->result;
      f32_team_sync<kTW>(team);                          // nobody reads the scratch after this point
      return r;
    }
    // too many elements in the bin: split its value range again
    float mn = __int_as_float(0x7f800000), mx = __int_as_float(0xff800000);
    for (int i = tl; i < n; i += TT) {
      const float v = x[i];
      if (f32_bin(v, vlo, scale) == beta) { mn = fminf(mn, v); mx = fmaxf(mx, v); }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      mn = fminf(mn, __shfl_xor_sync(FULL, mn, o));
      mx = fmaxf(mx, __shfl_xor_sync(FULL, mx, o));
    }
    if (kTW > 1) {
      const int wt = tl >> 5;
      if (lane == 0) { T->red[0][wt][0] = (double)mn; T->red[0][wt][1] = (double)mx; }
      f32_team_sync<kTW>(team);
#pragma unroll
      for (int w = 0; w < kTW; ++w) { mn = fminf(mn, (float)T->red[0][w][0]); mx = fmaxf(mx, (float)T->red[0][w][1]); }
      f32_team_sync<kTW>(team);
    }
    if (mn == mx) return mn;
    vlo = mn;
    scale = 255.5f / (mx - mn);
    if (!(scale < 1e30f)) break;                         // range too small for float arithmetic: bisection
  }
  // last resort: bisection on the order-preserving keys, 32 counting passes (always terminates)
  uint32_t klo = 0u, khi = 0xffffffffu;                  // smallest key with count(key <= .) > rho lies in [klo, khi]
  int sel = 0;
  while (klo < khi) {
    const uint32_t mid = klo + ((khi - klo) >> 1);
    uint32_t cnt = 0;
    for (int i = tl; i < n; i += TT) cnt += f32_key(x[i]) <= mid;
    cnt = __reduce_add_sync(FULL, cnt);
    if (kTW > 1) {
      const int wt = tl >> 5;
      if (lane == 0) T->redu[sel][wt][1] = cnt;
      f32_team_sync<kTW>(team);
      cnt = 0;
#pragma unroll
      for (int w = 0; w < kTW; ++w) cnt += T->redu[sel][w][1];
      sel ^= 1;
    }
    if (cnt > (uint32_t)rho) khi = mid; else klo = mid + 1;
  }
  const uint32_t b = (klo & 0x80000000u) ? (klo & 0x7fffffffu) : ~klo;
  return __int_as_float((int)b);
}

// ------------------------------------------------------------------------------------------------
// One window, all thresholds, by one team.  x points at the window (shared or global memory).
// ------------------------------------------------------------------------------------------------
template <int kTW>
__device__ __forceinline__ void f32_window(float* x, int n, const TdF32Params& P, uint8_t* flags, F32Team* T, int tl,
                                           int lane, int team) {
  constexpr int TT = 32 * kTW;
  const int wt = tl >> 5;
  int sel = 0;
  // ---------------------------------------------------------------- T2: statistics around the pivot
  // A = sum (x - c), B = sum (x - c)^2, so mu = c + A/n and sigma^2 = B/n - (A/n)^2.  The subtraction cancels when
  // the pivot is far from the mean in units of sigma (an RFI spike at x[0]; or the mean has moved after a huge
  // sample was replaced): whenever sigma^2 < 1e-6 B/n -- more than six of the sixteen digits gone -- the sums are
  // taken again around the current mean, where |A/n| is rounding noise.  Relative error of sigma^2 <= ~1e-10.
  double c = (double)x[0];
  double A = 0.0, B = 0.0;
  const double rn = 1.0 / (double)n;
  auto sums = [&]() {
    double A0 = 0.0, B0 = 0.0, A1 = 0.0, B1 = 0.0;
    int i = tl;
    for (; i + TT < n; i += 2 * TT) {
      const double d0 = (double)x[i] - c, d1 = (double)x[i + TT] - c;
      A0 += d0; B0 = fma(d0, d0, B0);
      A1 += d1; B1 = fma(d1, d1, B1);
    }
    if (i < n) { const double d0 = (double)x[i] - c; A0 += d0; B0 = fma(d0, d0, B0); }
    A = A0 + A1; B = B0 + B1;
    f32_team_sum2<kTW>(A, B, T, sel, wt, lane, team);
  };
  auto cancels = [&]() {                                 // team-uniform
    const double am = A * rn, m2 = B * rn;
    return m2 - am * am < 1e-6 * m2;
  };
  sums();
  if (cancels()) { c += A * rn; sums(); }
  for (int it = 0; it < P.n_thr; ++it) {
    // ---------------------------------------------------------------- T3: bounds
    const double am = A * rn;
    const double mu = c + am;
    double var = B * rn - am * am;
    if (!(var > 0.0)) var = 0.0;
    const double sigma = sqrt(var);
    const double cut = P.k[it] * sigma;
    float t_lo, t_hi;
    f32_bounds(mu, cut, t_lo, t_hi);
    double dA = 0.0, dB = 0.0;
    uint32_t cnt = 0;
    if (P.policy == 0) {
      // ---------------------------------------------------------------- T4 (mean): one fused sweep
      const float r = (float)mu;
      const double dr = (double)r - c;
      for (int i = tl; i < n; i += TT) {
        const float v = x[i];
        if (v > t_hi || v < t_lo) {
          const double d = (double)v - c;
          dA += dr - d; dB += dr * dr - d * d;
          x[i] = r;
          ++cnt;
          if (flags) flags[i] = 1;
        }
      }
      cnt = f32_team_sum_u32<kTW>(cnt, T, sel, wt, lane, team);
      if (cnt == 0) continue;
    } else {
      // ---------------------------------------------------------------- T4 (median): detect, select, replace
      {
        uint32_t c0 = 0, c1 = 0;
        int i = tl;
        for (; i + TT < n; i += 2 * TT) {
          const float v0 = x[i], v1 = x[i + TT];
          c0 += (v0 > t_hi || v0 < t_lo);
          c1 += (v1 > t_hi || v1 < t_lo);
        }
        if (i < n) { const float v0 = x[i]; c0 += (v0 > t_hi || v0 < t_lo); }
        cnt = c0 + c1;
      }
      const uint32_t mine = cnt;
      cnt = f32_team_sum_u32<kTW>(cnt, T, sel, wt, lane, team);
      if (cnt == 0) continue;
      const float r = f32_team_median<kTW>(x, n, (float)mu, (float)sigma, T, tl, lane, team);
      if (mine) {
        const double dr = (double)r - c;
        for (int i = tl; i < n; i += TT) {
          const float v = x[i];
          if (v > t_hi || v < t_lo) {
            const double d = (double)v - c;
            dA += dr - d; dB += dr * dr - d * d;
            x[i] = r;
            if (flags) flags[i] = 1;
          }
        }
      }
    }
    if (it + 1 < P.n_thr) {
      f32_team_sum2<kTW>(dA, dB, T, sel, wt, lane, team);
      const double B_before = B;
      A += dA; B += dB;
      // sum again around the current mean when the update cannot be trusted: the mean has left the pivot behind, or
      // the replaced samples carried nearly all of B (a 1e8 sigma spike: B was 1e16 + the rest, in 53 bits)
      if (cancels() || B < 1e-6 * B_before) {
        f32_team_sync<kTW>(team);                        // every replacement of this iteration is visible
        c += A * rn;
        sums();
      }
    }
    if (tl == 0 && P.counts) atomicAdd(&P.counts[it], (unsigned long long)cnt);
  }
}

// dynamic shared memory: [seg_cap floats (16-byte multiple)] [teams x F32Team] [mbarrier]
template <int kTW>
__host__ __device__ constexpr int f32_teams() { return (kF32Threads / 32) / kTW; }

template <int kTW, bool kStage>
__global__ void __launch_bounds__(kF32Threads) td_f32_kernel(const TdF32Params P) {
  extern __shared__ __align__(128) uint8_t smem[];
  constexpr int NT = f32_teams<kTW>();
  const int seg_bytes = kStage ? ((P.seg * 4 + 15) & ~15) : 0;
  float* slot = reinterpret_cast<float*>(smem);
  F32Team* teams = reinterpret_cast<F32Team*>(smem + seg_bytes);
  uint64_t* bar = reinterpret_cast<uint64_t*>(smem + seg_bytes + NT * sizeof(F32Team));
  const int tid = threadIdx.x, lane = tid & 31;
  const int team = tid / (32 * kTW), tl = tid % (32 * kTW);
  F32Team* T = teams + team;
  if (kStage && tid == 0) {
    mbar_init(bar, 1);
    fence_mbar_init();
  }
  __syncthreads();
  uint32_t phase = 0;
  const int64_t units = P.rows * P.segs_per_row;
  for (int64_t u = blockIdx.x; u < units; u += gridDim.x) {
    const int64_t row = u / P.segs_per_row;
    const int s0 = (int)(u % P.segs_per_row) * P.seg;
    const int n = min(P.seg, P.S - s0);
    const float* g = P.src + row * P.stride + s0;
    float* go = P.dst + row * P.stride + s0;
    float* x;
    // ---------------------------------------------------------------- T1: load
    if (kStage) {
      x = slot;
      if (P.bulk) {
        const int nb = n & ~3;
        if (tid == 0 && nb > 0) {
          mbar_arrive_expect_tx(bar, (uint32_t)nb * 4u);
          bulk_load(slot, g, (uint32_t)nb * 4u, bar);
        }
        if (tid >= 32 && tid < 32 + (n - nb)) slot[nb + tid - 32] = g[nb + tid - 32];
        if (nb > 0) { mbar_wait(bar, phase); phase ^= 1; }
      } else {
        for (int i = tid; i < n; i += kF32Threads) slot[i] = g[i];
      }
    } else {
      x = go;
      if (go != g)
        for (int i = tid; i < n; i += kF32Threads) go[i] = g[i];
    }
    __syncthreads();
    // ---------------------------------------------------------------- T2..T5: windows of the segment
    const int nwin = (n + P.window - 1) / P.window;
    uint8_t* fl = P.flags ? P.flags + row * P.S + s0 : nullptr;
    for (int w = team; w < nwin; w += NT) {
      const int w0 = w * P.window;
      f32_window<kTW>(x + w0, min(P.window, n - w0), P, fl ? fl + w0 : nullptr, T, tl, lane, team);
    }
    // ---------------------------------------------------------------- T6: store
    if (kStage) {
      if (P.bulk) {
        fence_proxy_async_smem();
        __syncthreads();
        const int nb = n & ~3;
        if (tid == 0 && nb > 0) {
          bulk_store(go, slot, (uint32_t)nb * 4u);
          bulk_commit();
          bulk_wait_read<0>();
        }
        if (tid >= 32 && tid < 32 + (n - nb)) go[nb + tid - 32] = slot[nb + tid - 32];
      } else {
        __syncthreads();
        for (int i = tid; i < n; i += kF32Threads) go[i] = slot[i];
      }
    }
    __syncthreads();
  }
  if (kStage && P.bulk && tid == 0) bulk_wait_all<0>();
}

}  // namespace rfim
