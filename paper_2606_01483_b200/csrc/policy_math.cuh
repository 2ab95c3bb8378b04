// Closed form of the hybrid eviction policy, shared by the device kernels and the host-side
// mirror (argument validation / page accounting).  Product code: NOT shared with oracle/.
//
// Alg. 1 on the output region, Eq. 2 / Alg. 2 on the
// speech region, system prompts always kept.  Readings: DESIGN.md.
#pragma once
#include <stdint.h>

#ifdef __CUDACC__
#define MM_HD __host__ __device__ __forceinline__
#else
#define MM_HD inline
#endif

namespace murmur {

struct SeqParams {      // one sequence's regions, policy and fill level
  int32_t P, S, M;      // prefix / speech / mid sizes
  int32_t len;          // tokens appended so far
  int32_t w_s, d, k_s;  // speech window, delay, speech sinks
  int32_t w_o, k_o;     // output window, output sinks
};

struct Interval {
  int32_t a, b;  // [a, b)
};

MM_HD int32_t mm_min(int32_t x, int32_t y) { return x < y ? x : y; }
MM_HD int32_t mm_max(int32_t x, int32_t y) { return x > y ? x : y; }

// t: output tokens in the cache including the newest (0 while prefilling).
MM_HD int32_t seq_t(const SeqParams& s) { return mm_max(0, s.len - (s.P + s.S + s.M)); }

// l(t) = min(max(0, t - d), max(0, S - w_s))   (Alg. 2 lines 1-4; parks at the end of speech)
MM_HD int32_t window_start(const SeqParams& s, int32_t t) {
  return mm_min(mm_max(0, t - s.d), mm_max(0, s.S - s.w_s));  // no overflow: all operands >= 0
}

// End (exclusive, region-relative, clipped to S) of the speech window; overflow-safe for WINDOW_OFF.
MM_HD int32_t window_end(const SeqParams& s, int32_t l) { return (s.w_s >= s.S - l) ? s.S : l + s.w_s; }

// Maximal intervals of the retained set A(t) in absolute positions, clipped to [0, len).
// At most 6 before merging.  Returns the count.
MM_HD int retained_runs(const SeqParams& s, Interval out[6]) {
  const int32_t t = seq_t(s);
  const int32_t l = window_start(s, t);
  const int32_t B = s.P + s.S + s.M;
  Interval raw[6];
  raw[0] = {0, s.P};                                                    // prefix prompt
  raw[1] = {s.P, s.P + mm_min(s.k_s, s.S)};                             // speech sinks (Eq. 2)
  raw[2] = {s.P + mm_min(l, s.S), s.P + window_end(s, mm_min(l, s.S))};  // speech window (Alg. 2)
  raw[3] = {s.P + s.S, B};                                              // second prompt
  raw[4] = {B, B + mm_min(s.k_o, t)};                                   // output sinks (Alg. 1)
  raw[5] = {B + mm_max(0, t - mm_min(s.w_o, t)), B + t};                // last w_o outputs
  int n = 0;
  for (int i = 0; i < 6; ++i) {
    int32_t a = raw[i].a, b = mm_min(raw[i].b, s.len);
    if (b <= a) continue;
    if (n > 0 && a <= out[n - 1].b) {  // overlaps or touches the previous run: merge
      out[n - 1].b = mm_max(out[n - 1].b, b);
    } else {
      out[n].a = a;
      out[n].b = b;
      ++n;
    }
  }
  return n;
}

// Dead intervals (positions that can never be attended again) in absolute positions: speech
// behind the window that are not sinks, outputs behind the output window that are not sinks.
// At most 2; merged when adjacent.  Returns the count.
MM_HD int dead_intervals(const SeqParams& s, Interval out[2]) {
  const int32_t t = seq_t(s);
  const int32_t l = window_start(s, t);
  const int32_t B = s.P + s.S + s.M;
  int n = 0;
  const int32_t sa = s.P + mm_min(s.k_s, s.S), sb = mm_min(s.P + mm_min(l, s.S), s.len);
  if (sb > sa) {
    out[n].a = sa;
    out[n].b = sb;
    ++n;
  }
  const int32_t oa = B + mm_min(s.k_o, t), ob = mm_min(B + t - mm_min(s.w_o, t), s.len);
  if (ob > oa) {
    if (n > 0 && out[n - 1].b == oa) {
      out[n - 1].b = ob;
    } else {
      out[n].a = oa;
      out[n].b = ob;
      ++n;
    }
  }
  return n;
}

// Blocks (of p positions) lying completely inside [iv.a, iv.b): [lo, hi).
MM_HD void blocks_inside(const Interval& iv, int32_t p, int32_t* lo, int32_t* hi) {
  *lo = (iv.a + p - 1) / p;
  *hi = iv.b / p;
  if (*hi < *lo) *hi = *lo;
}

// Same for p = 2^plog (device code: no integer division on the step's critical path).
MM_HD void blocks_inside_log2(const Interval& iv, int32_t plog, int32_t* lo, int32_t* hi) {
  *lo = (iv.a + (1 << plog) - 1) >> plog;
  *hi = iv.b >> plog;
  if (*hi < *lo) *hi = *lo;
}

// Number of blocks that are dead (hence freed by an evict) when the policy is applied at the
// current fill level.
MM_HD int32_t dead_block_count(const SeqParams& s, int32_t p) {
  Interval iv[2];
  const int n = dead_intervals(s, iv);
  int32_t c = 0;
  for (int i = 0; i < n; ++i) {
    int32_t lo, hi;
    blocks_inside(iv[i], p, &lo, &hi);
    c += hi - lo;
  }
  return c;
}

MM_HD int32_t retained_count(const SeqParams& s) {
  Interval r[6];
  const int n = retained_runs(s, r);
  int32_t c = 0;
  for (int i = 0; i < n; ++i) c += r[i].b - r[i].a;
  return c;
}

}  // namespace murmur
