// td_f32_fast.cuh -- time-domain sigma cut (TDSC, Fig. 2) for float32 dynamic spectra with statistics
// windows and mean / lower-median replacement (BASELINE.json configs[4]): the tuned kernel for rows
// that fit shared memory and windows that are multiples of 4 samples (td_f32.cuh keeps every other request).
//
// What the ncu captures of td_f32_kernel showed (profiles/r2a_f32_*): 110 - 130 thread instructions per sample, i.e.
// the kernel was bound by its own instruction count -- scalar strided loops (8 instructions per element and pass),
// about ten passes per window for the median (a 258-bin histogram with shared-memory atomics, a compaction pass, a
// ranking), and for short windows a per-window scalar chain (fp64 square root, bounds, reductions) executed by all
// 32 lanes of a warp for 8 elements each.  This kernel does the same arithmetic with a third of the instructions:
//   T1  one CTA of 256 threads stages a whole row by one 1-D TMA bulk copy (as before).
//   --  a window is owned by a TEAM of G lanes, G in {4, 16, 64, 256} chosen on the host so that a lane holds at most
//       32 quads (16 for the config-5 windows) and all 256 threads have work: W = 256 -> 4 lanes (8 windows per
//       warp side by side, each with its own scalar chain), W = 1024 -> 16, the whole row -> the CTA.  Teams of a
//       warp diverge freely: every shuffle carries the team's own lane mask.
//   T2  one pass of 128-bit shared-memory loads; fp64 sums around a pivot, re-taken around the mean whenever the
//       subtraction sigma^2 = B/n - (A/n)^2 would lose more than six digits (td_f32.cuh has the argument).
//   T3  cut = k sigma in fp64 -> two float bounds that reproduce the fp64 test exactly (f32_bounds).
//   T4  detection pass: FMNMX over a quad, two compares per quad, a bit per flagged quad; the replacement pass visits
//       the flagged quads only.
//   T2m lower median by BRACKETING: counting passes with two pivots (from mu, sigma, then by interpolation) shrink
//       the value interval that holds rank (n-1)/2 to at most 32 elements, which are gathered (as 16-bit indices)
//       and ranked.  And it is taken at most ONCE per window: replacing samples by the lower median m never changes
//       the lower median -- with L samples < m and E samples = m (L <= rank < L + E), moving l samples from below
//       and u from above onto m gives L - l <= rank < L + E + u -- so every later iteration's snapshot median is m.
//   T5  statistics of the next iteration from the fp64 deltas of the replaced samples.   T6  one TMA bulk store.
#pragma once

#include "common.cuh"
#include "td_f32.cuh"   // TdF32Params, f32_bounds, f32_key

namespace rfim {

constexpr int kF32FastThreads = 256;
constexpr int kF32FastListCap = 32;    // capacity of a team's gather list (f32f_cap<G>() <= this)

// scratch of one team in shared memory
struct __align__(8) F32FastTeam {
  uint16_t list[kF32FastListCap];   // gathered candidates: element indices inside the window
  int ln;                           // gather cursor
  float result;
  int rec;                          // CTA-wide median search: this team's entry in the request list
  int pad;
};
// CTA-wide median search (one window per team and row): a request per window that needs its median
struct __align__(8) F32FastSel { int w0, n; float mu, sig, result; int pad; };
// exchange area of the teams that span several warps (G >= 64): at most 4 teams x 8 warps
struct __align__(16) F32FastXchg {
  double red[2][8][2];
  uint32_t redu[2][8];
  uint16_t biglist[64];             // gather list of a wide team (f32f_cap<G>() = 64 for G >= 64)
};
__host__ __device__ constexpr int f32_fast_teams(int G) { return kF32FastThreads / G; }
__host__ __device__ inline size_t f32_fast_smem_bytes(int S, int G) {
  size_t b = ((size_t)S * 4 + 15) & ~(size_t)15;
  b += (size_t)f32_fast_teams(G) * sizeof(F32FastTeam);
  if (G > 32) b = ((b + 15) & ~(size_t)15) + (size_t)f32_fast_teams(G) * sizeof(F32FastXchg);
  b = ((b + 15) & ~(size_t)15) + (size_t)f32_fast_teams(G) * sizeof(F32FastSel) + 16;   // requests + two counters
  return b + 16;
}

template <int G>
struct F32FastCtx {
  F32FastTeam* T;
  F32FastXchg* X;     // G > 32 only
  uint32_t tmask;     // lanes of this team inside its warp (G <= 32), else FULL
  int j;              // lane index inside the team
  int team;           // team index inside the CTA
  int lane, wt;       // lane inside the warp, warp inside the team
  int sel;            // exchange buffer
  // CTA-wide median search
  F32FastTeam* teams; // scratch of team 0
  F32FastSel* req;    // request list
  int* nreq;          // two counters, used alternately
  const float* slot;  // the staged row
  int ncall;          // calls so far (CTA-uniform)
};

template <int G>
__device__ __forceinline__ void f32f_sync(const F32FastCtx<G>& c) {
  if (G <= 32) __syncwarp(c.tmask);
  else if (G == kF32FastThreads) __syncthreads();
  else asm volatile("bar.sync %0, %1;" ::"r"(c.team + 1), "n"(G) : "memory");
}
template <int G>
__device__ __forceinline__ void f32f_sum2(double& a, double& b, F32FastCtx<G>& c) {
  constexpr int W = G < 32 ? G : 32;
#pragma unroll
  for (int o = W / 2; o > 0; o >>= 1) {
    a += __shfl_xor_sync(c.tmask, a, o);
    b += __shfl_xor_sync(c.tmask, b, o);
  }
  if (G > 32) {
    if (c.lane == 0) { c.X->red[c.sel][c.wt][0] = a; c.X->red[c.sel][c.wt][1] = b; }
    f32f_sync<G>(c);
    a = 0.0; b = 0.0;
#pragma unroll
    for (int w = 0; w < G / 32; ++w) { a += c.X->red[c.sel][w][0]; b += c.X->red[c.sel][w][1]; }
    c.sel ^= 1;
  }
}
template <int G>
__device__ __forceinline__ uint32_t f32f_sum_u32(uint32_t a, F32FastCtx<G>& c) {
  constexpr int W = G < 32 ? G : 32;
  if (W == 32) {
    a = __reduce_add_sync(FULL, a);
  } else {
#pragma unroll
    for (int o = W / 2; o > 0; o >>= 1) a += __shfl_xor_sync(c.tmask, a, o);
  }
  if (G > 32) {
    if (c.lane == 0) c.X->redu[c.sel][c.wt] = a;
    f32f_sync<G>(c);
    a = 0;
#pragma unroll
    for (int w = 0; w < G / 32; ++w) a += c.X->redu[c.sel][w];
    c.sel ^= 1;
  }
  return a;
}

// 0xFFFFFFFF if v <= p else 0 (one FSET; false for NaN).  Counting with these masks -- c -= m0 + m1 -- costs 1.5
// instructions per compare; `c += (v <= p)` compiles to a compare, an add and a predicated move on one dependent chain.
__device__ __forceinline__ uint32_t f32f_le_mask(float v, float p) {
  uint32_t m;
  asm("set.le.u32.f32 %0, %1, %2;" : "=r"(m) : "f"(v), "f"(p));
  return m;
}

// A lane's quads of a window of nq quads: j, j + G, ..., j + G (T - 1).  They are visited in the rotated order t0,
// t0 + 1, ..., T - 1, 0, ..., t0 - 1, so that the teams sharing a quarter-warp read different bank groups (G < 8
// only).  body(quad index, t).
struct F32Quads { int T, t0; };
template <int G, typename F>
__device__ __forceinline__ void f32f_each_quad(const F32Quads& q, int j, F&& body) {
  if (G < 8) {
#pragma unroll 2
    for (int t = q.t0; t < q.T; ++t) body(j + G * t, t);
    for (int t = 0; t < q.t0; ++t) body(j + G * t, t);
  } else {
#pragma unroll 2
    for (int t = 0; t < q.T; ++t) body(j + G * t, t);
  }
}
// elements a team gathers and ranks at the end of the median search: the ranking costs m^2 / G compares per lane
template <int G>
__host__ __device__ constexpr int f32f_cap() { return G <= 4 ? 12 : (G <= 16 ? 16 : (G <= 32 ? 32 : 64)); }

// Teams narrower than a warp run side by side in one warp.  Their heavy loops must stay CONVERGED (a warp that
// splits into its teams executes every loop once per team), so the control flow around them is warp-uniform: every
// lane of the warp takes part, a team that has nothing to do makes zero trips, and loop conditions are votes.
template <int G>
__device__ __forceinline__ bool f32f_any(bool p) {
  return G < 32 ? __any_sync(FULL, p) : p;             // G >= 32: the team owns its warps, p is team-uniform
}

// T2m: lower median (rank (n-1)/2 of the ascending values) of the window x4[0 .. n/4), by the whole team; every
// lane of a team with `need` returns it (teams without `need` just keep the warp together).  mu / sigma (floats)
// only guide the first pivots.  The values are only read.
template <int G>
__device__ float f32f_median(const float4* x4, int n, const F32Quads& Q, float muf, float sigf, bool need,
                             F32FastCtx<G>& c) {
  constexpr uint32_t CAP = (uint32_t)f32f_cap<G>();
  // Wide teams gather up to 64 candidates: with n = 12500 the second counting pass leaves 36 +- 6 of them, and a cap
  // of 32 meant a third pass over the row nearly every time.
  uint16_t* const list = G > 32 ? c.X->biglist : c.T->list;
  const float* x = reinterpret_cast<const float*>(x4);
  const uint32_t rho = need ? (uint32_t)(n - 1) >> 1 : 0u;
  const float inf = __int_as_float(0x7f800000);
  // invariant: #{v <= a} = ca <= rho < cb = #{v <= b}; the answer is the (rho - ca)-th smallest value in (a, b]
  float a = -inf, b = inf;
  uint32_t ca = 0, cb = need ? (uint32_t)n : 0u;
  // first pivots: the median of n Gaussian draws is within 1.25 sigma / sqrt(n) (one standard deviation) of mu
  float R = 3.2f * sigf * rsqrtf((float)max(n, 1));
  float p1 = muf - R, p2 = muf + R;
  bool done = !need;                                     // result known without gathering
  float result = 0.0f;
  bool searching = need && cb - ca > CAP;
  for (int pass = 0; pass < 64 && f32f_any<G>(searching); ++pass) {
    if (!(p1 > a)) p1 = a;                               // keep the pivots inside the bracket (also rejects NaN)
    if (!(p2 < b)) p2 = b;
    if (!(p1 <= p2)) p1 = p2;
    uint32_t c1 = 0, c2 = 0;                             // #{v <= p1}, #{v <= p2}
    uint32_t c1a = 0, c1b = 0, c2a = 0, c2b = 0;
    F32Quads Qs = Q;
    if (!searching) { Qs.T = 0; Qs.t0 = 0; }
    f32f_each_quad<G>(Qs, c.j, [&](int qi, int) {
      const float4 v = x4[qi];
      c1a -= f32f_le_mask(v.x, p1) + f32f_le_mask(v.y, p1);
      c1b -= f32f_le_mask(v.z, p1) + f32f_le_mask(v.w, p1);
      c2a -= f32f_le_mask(v.x, p2) + f32f_le_mask(v.y, p2);
      c2b -= f32f_le_mask(v.z, p2) + f32f_le_mask(v.w, p2);
    });
    c1 = c1a + c1b; c2 = c2a + c2b;
    // one reduction for both counts: n <= 2^15 in this kernel (the host checks), so each fits 16 bits
    const uint32_t packed = f32f_sum_u32<G>(c1 | (c2 << 16), c);
    if (searching) {
      c1 = packed & 0xffffu;
      c2 = packed >> 16;
      if (rho < c1) { b = p1; cb = c1; }
      else if (rho < c2) { a = p1; ca = c1; b = p2; cb = c2; }
      else { a = p2; ca = c2; }
      const uint32_t m = cb - ca;
      if (m <= CAP) {
        searching = false;
      } else if (a > -inf && b < inf) {
        // interpolate the rank inside (a, b] and step aside by a margin of a few binomial standard deviations
        const float w = b - a;
        const float f = ((float)(rho - ca) + 0.5f) / (float)m;
        const float dev = (2.0f * sqrtf(f * (1.0f - f) * (float)m) + 1.0f) / (float)m;
        p1 = a + w * fmaxf(f - dev, 0.0f);
        p2 = a + w * fminf(f + dev, 1.0f);
        if (!(p1 > a)) p1 = f32_next_up(a);              // the float grid is exhausted towards a
        if (!(p2 < b)) p2 = f32_next_down(b);
        if (!(p2 >= p1)) p2 = p1;
        if (!(w <= 3.0e38f)) {                           // (unreachable for |x| < 1e18) -> key bisection below
          searching = false;
        } else if (!(p1 < b)) {                          // a and b are neighbouring floats: every value in (a, b] is b
          searching = false; done = true; result = b;
        }
      } else if (b == inf && a == -inf) {                // (both pivots collapsed: cannot happen, but stay finite)
        R *= 2.0f;
        p1 = muf - R; p2 = muf + R;
      } else if (b == inf) {                             // everything seen so far lies below the rank: go up
        R *= 4.0f;
        p1 = a + R; p2 = a + 4.0f * R;
        if (!(p1 > a)) { p1 = 3.402823466e38f; p2 = 3.402823466e38f; }
        if (!(p2 < inf)) p2 = 3.402823466e38f;
      } else {                                           // a == -inf: go down
        R *= 4.0f;
        p2 = b - R; p1 = b - 4.0f * R;
        if (!(p2 < b)) { p1 = -3.402823466e38f; p2 = -3.402823466e38f; }
        if (!(p1 > -inf)) p1 = -3.402823466e38f;
      }
    }
  }
  // last resort (the bracket did not shrink in 64 passes: a pathological value distribution): bisection on the
  // order-preserving integer keys, 32 counting passes, always terminates
  bool bisect = need && !done && cb - ca > CAP;
  if (f32f_any<G>(bisect)) {
    uint32_t klo = 0u, khi = 0xffffffffu;
    for (int step = 0; step < 32; ++step) {              // 32 halvings of a 2^32 range
      const uint32_t mid = klo + ((khi - klo) >> 1);
      uint32_t cnt = 0;
      F32Quads Qs = Q;
      if (!bisect) { Qs.T = 0; Qs.t0 = 0; }
      f32f_each_quad<G>(Qs, c.j, [&](int qi, int) {
        const float4 v = x4[qi];
        cnt += (f32_key(v.x) <= mid) + (f32_key(v.y) <= mid) + (f32_key(v.z) <= mid) + (f32_key(v.w) <= mid);
      });
      cnt = f32f_sum_u32<G>(cnt, c);
      if (cnt > rho) khi = mid; else klo = mid + 1;
    }
    if (bisect) {
      const uint32_t bits = (klo & 0x80000000u) ? (klo & 0x7fffffffu) : ~klo;
      result = __int_as_float((int)bits);
      done = true;
    }
  }
  // gather the (at most CAP) elements of (a, b] as indices, then rank them: the one with rank rho - ca is the median
  const bool gather = need && !done;
  const uint32_t m = gather ? cb - ca : 0u;
  if (c.j == 0) c.T->ln = 0;
  f32f_sync<G>(c);
  {
    F32Quads Qs = Q;
    if (!gather) { Qs.T = 0; Qs.t0 = 0; }
    f32f_each_quad<G>(Qs, c.j, [&](int qi, int) {
      const float4 v = x4[qi];
      const bool in0 = v.x > a && v.x <= b, in1 = v.y > a && v.y <= b, in2 = v.z > a && v.z <= b, in3 = v.w > a && v.w <= b;
      if (in0 | in1 | in2 | in3) {
        if (in0) list[atomicAdd(&c.T->ln, 1)] = (uint16_t)(4 * qi);
        if (in1) list[atomicAdd(&c.T->ln, 1)] = (uint16_t)(4 * qi + 1);
        if (in2) list[atomicAdd(&c.T->ln, 1)] = (uint16_t)(4 * qi + 2);
        if (in3) list[atomicAdd(&c.T->ln, 1)] = (uint16_t)(4 * qi + 3);
      }
    });
  }
  f32f_sync<G>(c);
  const uint32_t want = rho - ca;
  for (uint32_t i = (uint32_t)c.j; i < m; i += G) {
    const uint32_t ii = list[i];
    const float e = x[ii];
    uint32_t rank = 0;
    for (uint32_t k = 0; k < m; ++k) {
      const uint32_t kk = list[k];
      const float o = x[kk];
      rank += (o < e) || (o == e && kk < ii);
    }
    if (rank == want) c.T->result = e;
  }
  f32f_sync<G>(c);
  if (gather) result = c.T->result;
  f32f_sync<G>(c);                                       // nobody reads the scratch after this point
  return result;
}

// The same search by a team of Gv lanes chosen at run time (4 <= Gv <= 32, lanes vmask of one warp); every warp of
// the CTA calls it together, teams without a window (act = false) only keep their warp converged.
__device__ inline float f32f_median_rt(const float4* x4, int n, int jv, int Gv, uint32_t vmask, F32FastTeam* T, float muf,
                                float sigf, bool act) {
  const float* x = reinterpret_cast<const float*>(x4);
  // Gathering m candidates and ranking them costs about 5 m^2 / Gv instructions per lane, one more counting pass about
  // 3.5 n / Gv: the cap follows the window length (after the second pass m is 15 +- 4 for n = 256, 20 +- 4.5 for 1024;
  // measured: W = 1024 0.734 -> 0.727 ms with 26 instead of 16, W = 256 best with 12 / 16)
  const uint32_t CAP = n <= 256 ? (Gv <= 4 ? 12u : 16u) : (n <= 1024 ? 26u : 32u);
  const int nq = act ? n >> 2 : 0;
  const uint32_t rho = act ? (uint32_t)(n - 1) >> 1 : 0u;
  const float inf = __int_as_float(0x7f800000);
  auto sum_u32 = [&](uint32_t v) {
    for (int o = Gv >> 1; o > 0; o >>= 1) v += __shfl_xor_sync(vmask, v, o);
    return v;
  };
  float a = -inf, b = inf;
  uint32_t ca = 0, cb = act ? (uint32_t)n : 0u;
  float R = 3.2f * sigf * rsqrtf((float)max(n, 1));
  float p1 = muf - R, p2 = muf + R;
  bool done = !act;
  float result = 0.0f;
  bool searching = act && cb - ca > CAP;
  for (int pass = 0; pass < 64 && __any_sync(FULL, searching); ++pass) {
    if (!(p1 > a)) p1 = a;
    if (!(p2 < b)) p2 = b;
    if (!(p1 <= p2)) p1 = p2;
    uint32_t c1a = 0, c1b = 0, c2a = 0, c2b = 0;
    const int nqs = searching ? nq : 0;
#pragma unroll 2
    for (int qi = jv; qi < nqs; qi += Gv) {
      const float4 v = x4[qi];
      c1a -= f32f_le_mask(v.x, p1) + f32f_le_mask(v.y, p1);
      c1b -= f32f_le_mask(v.z, p1) + f32f_le_mask(v.w, p1);
      c2a -= f32f_le_mask(v.x, p2) + f32f_le_mask(v.y, p2);
      c2b -= f32f_le_mask(v.z, p2) + f32f_le_mask(v.w, p2);
    }
    const uint32_t packed = sum_u32((c1a + c1b) | ((c2a + c2b) << 16));
    if (searching) {
      const uint32_t c1 = packed & 0xffffu, c2 = packed >> 16;
      if (rho < c1) { b = p1; cb = c1; }
      else if (rho < c2) { a = p1; ca = c1; b = p2; cb = c2; }
      else { a = p2; ca = c2; }
      const uint32_t m = cb - ca;
      if (m <= CAP) {
        searching = false;
      } else if (a > -inf && b < inf) {
        const float w = b - a;
        const float f = ((float)(rho - ca) + 0.5f) / (float)m;
        const float dev = (2.0f * sqrtf(f * (1.0f - f) * (float)m) + 1.0f) / (float)m;
        p1 = a + w * fmaxf(f - dev, 0.0f);
        p2 = a + w * fminf(f + dev, 1.0f);
        if (!(p1 > a)) p1 = f32_next_up(a);
        if (!(p2 < b)) p2 = f32_next_down(b);
        if (!(p2 >= p1)) p2 = p1;
        if (!(w <= 3.0e38f)) searching = false;
        else if (!(p1 < b)) { searching = false; done = true; result = b; }
      } else if (b == inf && a == -inf) {
        R *= 2.0f;
        p1 = muf - R; p2 = muf + R;
      } else if (b == inf) {
        R *= 4.0f;
        p1 = a + R; p2 = a + 4.0f * R;
        if (!(p1 > a)) { p1 = 3.402823466e38f; p2 = 3.402823466e38f; }
        if (!(p2 < inf)) p2 = 3.402823466e38f;
      } else {
        R *= 4.0f;
        p2 = b - R; p1 = b - 4.0f * R;
        if (!(p2 < b)) { p1 = -3.402823466e38f; p2 = -3.402823466e38f; }
        if (!(p1 > -inf)) p1 = -3.402823466e38f;
      }
    }
  }
  const bool bisect = act && !done && cb - ca > CAP;
  if (__any_sync(FULL, bisect)) {
    uint32_t klo = 0u, khi = 0xffffffffu;
    for (int step = 0; step < 32; ++step) {
      const uint32_t mid = klo + ((khi - klo) >> 1);
      uint32_t cnt = 0;
      const int nqs = bisect ? nq : 0;
      for (int qi = jv; qi < nqs; qi += Gv) {
        const float4 v = x4[qi];
        cnt += (f32_key(v.x) <= mid) + (f32_key(v.y) <= mid) + (f32_key(v.z) <= mid) + (f32_key(v.w) <= mid);
      }
      cnt = sum_u32(cnt);
      if (cnt > rho) khi = mid; else klo = mid + 1;
    }
    if (bisect) {
      const uint32_t bits = (klo & 0x80000000u) ? (klo & 0x7fffffffu) : ~klo;
      result = __int_as_float((int)bits);
      done = true;
    }
  }
  const bool gather = act && !done;
  const uint32_t m = gather ? cb - ca : 0u;
  if (act && jv == 0) T->ln = 0;
  __syncwarp(vmask);
  {
    const int nqs = gather ? nq : 0;
    for (int qi = jv; qi < nqs; qi += Gv) {
      const float4 v = x4[qi];
      const bool in0 = v.x > a && v.x <= b, in1 = v.y > a && v.y <= b, in2 = v.z > a && v.z <= b, in3 = v.w > a && v.w <= b;
      if (in0 | in1 | in2 | in3) {
        if (in0) T->list[atomicAdd(&T->ln, 1)] = (uint16_t)(4 * qi);
        if (in1) T->list[atomicAdd(&T->ln, 1)] = (uint16_t)(4 * qi + 1);
        if (in2) T->list[atomicAdd(&T->ln, 1)] = (uint16_t)(4 * qi + 2);
        if (in3) T->list[atomicAdd(&T->ln, 1)] = (uint16_t)(4 * qi + 3);
      }
    }
  }
  __syncwarp(vmask);
  const uint32_t want = rho - ca;
  for (uint32_t i = (uint32_t)jv; i < m; i += (uint32_t)Gv) {
    const uint32_t ii = T->list[i];
    const float e = x[ii];
    uint32_t rank = 0;
    for (uint32_t k = 0; k < m; ++k) {
      const uint32_t kk = T->list[k];
      const float o = x[kk];
      rank += (o < e) || (o == e && kk < ii);
    }
    if (rank == want) T->result = e;
  }
  __syncwarp(vmask);
  if (gather) result = T->result;
  __syncwarp(vmask);
  return result;
}

// CTA-wide median search (every thread of the CTA calls it): the windows that need their median are listed, the
// 256 lanes are re-divided evenly among them (32, 16, 8 or 4 lanes per window), each such team runs the search on
// its window, and the owners pick their result up.  Half the windows of a row need no median at k = 3: this keeps
// every lane busy during the search instead of every second team.
template <int G>
__device__ float f32f_cta_median(int w0, int n, float muf, float sigf, bool need, F32FastCtx<G>& c) {
  const int tid = threadIdx.x;
  int* const cnt = &c.nreq[c.ncall & 1];
  if (need && c.j == 0) {
    const int my = atomicAdd(cnt, 1);
    F32FastSel r;
    r.w0 = w0; r.n = n; r.mu = muf; r.sig = sigf; r.result = 0.0f; r.pad = 0;
    c.req[my] = r;
    c.T->rec = my;
  }
  __syncthreads();
  if (tid == 0) c.nreq[(c.ncall + 1) & 1] = 0;         // the counter of the previous call: everybody is past it
  ++c.ncall;
  const int K = *cnt;
  int Gv = 32;
  while (Gv * K > kF32FastThreads) Gv >>= 1;           // K <= 256 / G <= 64, so Gv >= 4
  const int v = tid / Gv, jv = tid % Gv;
  const bool act = v < K;
  const F32FastSel r = c.req[act ? v : 0];
  const uint32_t vmask = Gv == 32 ? FULL : (((1u << Gv) - 1u) << (c.lane & ~(Gv - 1)));
  const float med = f32f_median_rt(reinterpret_cast<const float4*>(c.slot + r.w0), r.n, jv, Gv, vmask,
                                   c.teams + (act ? v : 0), r.mu, r.sig, act);
  if (act && jv == 0) c.req[v].result = med;
  __syncthreads();
  return need ? c.req[c.T->rec].result : 0.0f;
}

// Warp-wide median search for teams narrower than a warp (every lane of the warp calls it): the windows of this
// warp's teams that need their median are counted by a ballot, the 32 lanes are re-divided evenly among them (32, 16,
// 8 or 4 lanes per window), each such team runs the search on its window, and the owners pick their result up by a
// shuffle.  At k = 3 only half of the W = 256 windows need a median: this keeps every lane busy during the search,
// with no barrier beyond the warp.
template <int G>
__device__ float f32f_warp_median(int w0, int n, float muf, float sigf, bool need, F32FastCtx<G>& c) {
  const int lane = c.lane;
  const uint32_t lead = __ballot_sync(FULL, need && c.j == 0);     // leaders of the teams that need a median
  const int K = __popc(lead);                                      // >= 1 (the caller voted)
  int Gv = 32;
  while (Gv * K > 32) Gv >>= 1;                                    // K <= 32 / G <= 8, so Gv >= 4
  const int v = lane / Gv, jv = lane % Gv;
  const bool act = v < K;
  const int src = (int)__fns(lead, 0, (act ? v : 0) + 1);          // leader lane of the window this lane works on
  const int w0v = __shfl_sync(FULL, w0, src), nv = __shfl_sync(FULL, n, src);
  const float muv = __shfl_sync(FULL, muf, src), sigv = __shfl_sync(FULL, sigf, src);
  const uint32_t vmask = Gv == 32 ? FULL : (((1u << Gv) - 1u) << (lane & ~(Gv - 1)));
  F32FastTeam* const Tv = c.T - (lane / G) + (src / G);            // scratch of the team that owns that window
  const float med = f32f_median_rt(reinterpret_cast<const float4*>(c.slot + w0v), nv, jv, Gv, vmask, Tv, muv, sigv, act);
  // the window of the team whose leader is lane l was served by virtual team number popc(lead below l)
  const int mine = __popc(lead & ((1u << (lane & ~(G - 1))) - 1u));
  const float out = __shfl_sync(FULL, med, mine * Gv);
  return need ? out : 0.0f;
}

// One window, all thresholds, by one team.  x4 points at the window in shared memory, n is a multiple of 4; a team
// without a window (valid = false: more teams than windows in this round) only keeps its warp together.
// kCta: every team of the CTA is inside this function at the same time (one window per team and row), so the median
// search may be CTA-wide.
template <int G, bool kCta>
__device__ __forceinline__ void f32f_window(float4* x4, int n, bool valid, const TdF32Params& P, uint8_t* flags,
                                            int team_in_warp, F32FastCtx<G>& c) {
  const int nq = valid ? n >> 2 : 0;
  F32Quads Q;
  Q.T = nq > c.j ? (nq - c.j + G - 1) / G : 0;
  Q.t0 = 0;
  if (G < 8 && Q.T > 0) Q.t0 = (team_in_warp & (8 / G - 1)) % Q.T;
  const float* xs = reinterpret_cast<const float*>(x4);
  // ---------------------------------------------------------------- T2: statistics around the pivot
  double piv = valid ? (double)xs[0] : 0.0;
  double A = 0.0, B = 0.0;
  const double rn = 1.0 / (double)(valid ? n : 1);
  auto sums = [&](bool mine) {
    double A0 = 0.0, B0 = 0.0, A1 = 0.0, B1 = 0.0;
    F32Quads Qs = Q;
    if (!mine) { Qs.T = 0; Qs.t0 = 0; }
    f32f_each_quad<G>(Qs, c.j, [&](int qi, int) {
      const float4 v = x4[qi];
      const double d0 = (double)v.x - piv, d1 = (double)v.y - piv, d2 = (double)v.z - piv, d3 = (double)v.w - piv;
      A0 += d0; B0 = fma(d0, d0, B0);
      A1 += d1; B1 = fma(d1, d1, B1);
      A0 += d2; B0 = fma(d2, d2, B0);
      A1 += d3; B1 = fma(d3, d3, B1);
    });
    double a2 = A0 + A1, b2 = B0 + B1;
    f32f_sum2<G>(a2, b2, c);
    if (mine) { A = a2; B = b2; }
  };
  auto cancels = [&]() {                                 // team-uniform
    const double am = A * rn, m2 = B * rn;
    return m2 - am * am < 1e-6 * m2;
  };
  sums(true);
  {
    const bool again = valid && cancels();
    if (f32f_any<G>(again)) {
      if (again) piv += A * rn;
      sums(again);
    }
  }

  bool have_median = false;
  float median = 0.0f;
  for (int it = 0; it < P.n_thr; ++it) {
    // ---------------------------------------------------------------- T3: bounds
    const double am = A * rn;
    const double mu = piv + am;
    double var = B * rn - am * am;
    if (!(var > 0.0)) var = 0.0;
    const double sigma = sqrt(var);
    const double cut = P.k[it] * sigma;
    float t_lo, t_hi;
    f32_bounds(mu, cut, t_lo, t_hi);
    // ---------------------------------------------------------------- T4: detect (a bit per flagged quad)
    uint32_t fm = 0;                                     // bit t <=> the lane's quad j + G t holds a flagged sample
    f32f_each_quad<G>(Q, c.j, [&](int qi, int t) {
      const float4 v = x4[qi];
      const float lo = fminf(fminf(v.x, v.y), fminf(v.z, v.w)), hi = fmaxf(fmaxf(v.x, v.y), fmaxf(v.z, v.w));
      if (hi > t_hi || lo < t_lo) fm |= 1u << t;
    });
    uint32_t cnt = 0;
    {
      uint32_t f2 = fm;
      while (f2) {
        const int t = __ffs(f2) - 1;
        f2 &= f2 - 1;
        const float4 v = x4[c.j + G * t];
        cnt += (v.x > t_hi || v.x < t_lo) + (v.y > t_hi || v.y < t_lo) + (v.z > t_hi || v.z < t_lo) +
               (v.w > t_hi || v.w < t_lo);
      }
    }
    cnt = f32f_sum_u32<G>(cnt, c);
    const bool flagged = cnt != 0;                       // team-uniform
    // ---------------------------------------------------------------- T2m / replacement value
    const bool need_med = flagged && P.policy != 0 && !have_median;
    if (kCta) {
      if (__syncthreads_or(need_med)) {
        const int w0 = (int)(reinterpret_cast<const float*>(x4) - c.slot);
        const float med = f32f_cta_median<G>(w0, n, (float)mu, (float)sigma, need_med, c);
        if (need_med) { median = med; have_median = true; }
      }
    } else if (f32f_any<G>(need_med)) {
      float med;
      if (G < 32) {
        med = f32f_warp_median<G>((int)(reinterpret_cast<const float*>(x4) - c.slot), n, (float)mu, (float)sigma, need_med, c);
      } else {
        med = f32f_median<G>(x4, n, Q, (float)mu, (float)sigma, need_med, c);
      }
      if (need_med) { median = med; have_median = true; }
    }
    const float r = P.policy == 0 ? (float)mu : median;
    // ---------------------------------------------------------------- T4: replace, T5: deltas
    double dA = 0.0, dB = 0.0;
    const double dr = (double)r - piv;
    while (fm) {
      const int t = __ffs(fm) - 1;
      fm &= fm - 1;
      const int qi = c.j + G * t;
      float4 v = x4[qi];
      float* pv = reinterpret_cast<float*>(&v);
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const float e = pv[u];
        if (e > t_hi || e < t_lo) {
          const double d = (double)e - piv;
          dA += dr - d; dB += dr * dr - d * d;
          pv[u] = r;
          if (flags) flags[4 * qi + u] = 1;
        }
      }
      x4[qi] = v;
    }
    if (it + 1 < P.n_thr && f32f_any<G>(flagged)) {
      f32f_sum2<G>(dA, dB, c);
      const double B_before = B;
      A += dA; B += dB;
      // sum again around the current mean when the update cannot be trusted: the mean has left the pivot behind, or
      // the replaced samples carried nearly all of B (a 1e8 sigma spike: B was 1e16 + the rest, in 53 bits)
      const bool again = flagged && (cancels() || B < 1e-6 * B_before);
      if (f32f_any<G>(again)) {
        f32f_sync<G>(c);                                 // the team's replacements are visible
        if (again) piv += A * rn;
        sums(again);
      }
    }
    if (flagged && c.j == 0 && P.counts) atomicAdd(&P.counts[it], (unsigned long long)cnt);
  }
}

// dynamic shared memory: [row: S floats][teams x F32FastTeam][G > 32: teams x F32FastXchg][mbarrier]
template <int G>
__global__ void __launch_bounds__(kF32FastThreads, 4) td_f32_fast_kernel(const TdF32Params P) {
  extern __shared__ __align__(128) uint8_t smem[];
  constexpr int NT = kF32FastThreads / G;
  const size_t row_bytes = ((size_t)P.S * 4 + 15) & ~(size_t)15;
  float* slot = reinterpret_cast<float*>(smem);
  F32FastTeam* teams = reinterpret_cast<F32FastTeam*>(smem + row_bytes);
  size_t off = row_bytes + (size_t)NT * sizeof(F32FastTeam);
  F32FastXchg* xchg = nullptr;
  if (G > 32) {
    off = (off + 15) & ~(size_t)15;
    xchg = reinterpret_cast<F32FastXchg*>(smem + off);
    off += (size_t)NT * sizeof(F32FastXchg);
  }
  off = (off + 15) & ~(size_t)15;
  F32FastSel* req = reinterpret_cast<F32FastSel*>(smem + off);
  off += (size_t)NT * sizeof(F32FastSel);
  int* nreq = reinterpret_cast<int*>(smem + off);
  off += 16;
  uint64_t* bar = reinterpret_cast<uint64_t*>(smem + ((off + 7) & ~(size_t)7));
  const int tid = threadIdx.x, lane = tid & 31;
  F32FastCtx<G> c;
  c.team = tid / G;
  c.j = tid % G;
  c.lane = lane;
  c.wt = (tid % G) >> 5;
  c.sel = 0;
  c.T = teams + c.team;
  c.X = G > 32 ? xchg + c.team : nullptr;
  c.tmask = G >= 32 ? FULL : (((1u << (G & 31)) - 1u) << (lane & ~(G - 1)));
  c.teams = teams; c.req = req; c.nreq = nreq; c.slot = slot; c.ncall = 0;
  if (tid < 2) nreq[tid] = 0;
  const int team_in_warp = G >= 32 ? 0 : (lane / G);
  if (tid == 0) {
    mbar_init(bar, 1);
    fence_mbar_init();
  }
  __syncthreads();
  uint32_t phase = 0;
  const int nwin = (P.S + P.window - 1) / P.window;
  for (int64_t row = blockIdx.x; row < P.rows; row += gridDim.x) {
    const float* g = P.src + row * P.stride;
    float* go = P.dst + row * P.stride;
    // ---------------------------------------------------------------- T1: load (S is a multiple of 4)
    if (tid == 0) {
      mbar_arrive_expect_tx(bar, (uint32_t)P.S * 4u);
      bulk_load(slot, g, (uint32_t)P.S * 4u, bar);
    }
    mbar_wait(bar, phase);
    phase ^= 1;
    // ---------------------------------------------------------------- T2..T5: windows of the row
    uint8_t* fl = P.flags ? P.flags + row * P.S : nullptr;
    if (G <= 4 && nwin <= NT && P.policy != 0) {
      // one window per team of 4 lanes (config 5, W = 256: 49 windows on 64 teams): the median search is CTA-wide.
      // (Teams of 16 lanes re-divide the lanes inside their warp instead -- W = 1024: 0.73 ms against 0.85 ms CTA-wide;
      // for teams of 4 it is the other way round, 0.87 against 0.83 ms.)
      const int w = c.team;
      const bool valid = w < nwin;
      const int w0 = valid ? w * P.window : 0;
      f32f_window<G, true>(reinterpret_cast<float4*>(slot + w0), valid ? min(P.window, P.S - w0) : 0, valid, P,
                           fl ? fl + w0 : nullptr, team_in_warp, c);
    } else {
      for (int wb = 0; wb < nwin; wb += NT) {           // a round of NT windows: warp-uniform trip count
        const int w = wb + c.team;
        const bool valid = w < nwin;
        if (G >= 32 && !valid) continue;                 // (a team of whole warps may simply skip)
        const int w0 = valid ? w * P.window : 0;
        f32f_window<G, false>(reinterpret_cast<float4*>(slot + w0), valid ? min(P.window, P.S - w0) : 0, valid, P,
                              fl ? fl + w0 : nullptr, team_in_warp, c);
      }
    }
    // ---------------------------------------------------------------- T6: store
    fence_proxy_async_smem();
    __syncthreads();
    if (tid == 0) {
      bulk_store(go, slot, (uint32_t)P.S * 4u);
      bulk_commit();
      bulk_wait_read<0>();
    }
    __syncthreads();
  }
  if (tid == 0) bulk_wait_all<0>();
}

}  // namespace rfim
