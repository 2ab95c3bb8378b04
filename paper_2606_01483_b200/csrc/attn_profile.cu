// murmur_attn_profile: the attention-sparsity profile of one decode step.
//
// PAPER.md:77 ("at any individual decode step, fewer than 25% of speech tokens account for 99% of
// attention weight") and the caption of Fig. 5: per query head, the FEWEST tokens of
// the KV cache whose Eq. 1 weights sum to >= frac of the total ("kept"), split
// into prompt / speech / text, next to the region totals ("evictable" = total - kept), plus the
// attention mass a candidate window policy would preserve (sum of weights inside its A(t)).
// It profiles the RESIDENT cache (every position that is not dead), so it is meant to be run on a
// cache kept without eviction (MURMUR_WINDOW_OFF) with the policy under study as the candidate.
//
// One CTA per (layer, sequence, KV head), 8 warps.
//   pass 1  warp per token: q . k for the G heads of the group with FFMA straight from the
//           (pre-swizzled) pool rows, fp32 -> scratch[h][x] (dead / unmapped positions: -inf)
//   pass 2  per head: M = max, e_x = exp(s_x - M) written back in place, L = sum e (fp64
//           accumulation), region masses and candidate coverage
//   pass 3  per head: the mass set has no sort - its threshold weight is found by bisection on the
//           bit pattern of e (non-negative floats order like unsigned integers): the largest tau with
//           sum{e >= tau} >= frac * L, 31 passes over L2-resident scratch.  Then
//           k = #{e > tau} + (as many of the ties at tau, in ascending position, as are needed).
#include <cuda_bf16.h>

#include <mutex>

#include "../../include/murmur.h"
#include "device_state.cuh"

// Built-in scratch of murmur_attn_profile_noalloc (see the end of this file and include/murmur.h).  It is part of
// the library image: every GPU that loads libmurmur.so sets these 8 MiB of its memory aside until the process
// exits, whether or not the call is ever made.  One array per GPU, shared by every handle, stream and thread.
// The name below is only usable as an address in DEVICE code; host code has to ask the runtime for the array's
// address on the current device (cudaGetSymbolAddress) - launch_attn_profile_noalloc does, once per device.
static __device__ __align__(256) unsigned char murmur_profile_builtin_scratch[MURMUR_PROFILE_NOALLOC_MAX_BYTES];

namespace murmur {
namespace {

constexpr int kProfWarps = 8;
constexpr int kProfThreads = kProfWarps * 32;

__device__ __forceinline__ float bf_lo(uint32_t w) { return __uint_as_float(w << 16); }
__device__ __forceinline__ float bf_hi(uint32_t w) { return __uint_as_float(w & 0xffff0000u); }

struct ProfParams {
  const uint16_t* q;
  murmur_profile_t* out;
  float* scratch;
  long long stride;  // floats per (CTA, head) row of scratch
  int seq_base, n_seqs_total, layer_begin;
  float sm_scale, frac;
  int use_candidate;
  uint8_t* member;  // optional [CTA][stride]: 1 where the position is in the mass set of any head of the group
  SeqParams cand;  // policy fields only (P, S, M, len are taken from the sequence)
};

// block-wide sums of up to 4 doubles (all threads get the result)
__device__ __forceinline__ void block_sum4(double (&v)[4], double (*sh)[4]) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
#pragma unroll
  for (int k = 0; k < 4; ++k)
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v[k] += __shfl_xor_sync(0xffffffffu, v[k], o);
  __syncthreads();
  if (lane == 0)
#pragma unroll
    for (int k = 0; k < 4; ++k) sh[warp][k] = v[k];
  __syncthreads();
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    double a = 0.0;
#pragma unroll
    for (int w = 0; w < kProfWarps; ++w) a += sh[w][k];
    v[k] = a;
  }
}

__device__ __forceinline__ int region_of(int x, int P, int S, int M) {  // 0 prompt, 1 speech, 2 text
  if (x < P) return 0;
  if (x < P + S) return 1;
  if (x < P + S + M) return 0;
  return 2;
}

__global__ void __launch_bounds__(kProfThreads)
attn_profile_kernel(const __grid_constant__ CacheView c, const __grid_constant__ SeqList list,
                    const __grid_constant__ ProfParams prm) {
  __shared__ float s_q[kMaxGroup][kHeadDim];
  __shared__ double s_red[kProfWarps][4];
  __shared__ int s_scan[kProfThreads + 1];
  __shared__ Interval s_cand[6];
  __shared__ int s_ncand;
  const int g = blockIdx.x, i = blockIdx.y, lc = blockIdx.z;
  const int layer = prm.layer_begin + lc;
  const int id = list.ids[i];
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int G = c.group, p = c.p, plog = c.p_log2;
  const SeqParams sp = load_params(c.seqs[id]);
  const int len = sp.len;
  Interval dead[2];
  const int n_dead = dead_intervals(sp, dead);
  const int32_t* tab = c.block_table + (size_t)id * c.max_blocks;
  const size_t cta = ((size_t)lc * gridDim.y + i) * gridDim.x + g;
  float* sc = prm.scratch + cta * (size_t)G * prm.stride;

  const size_t q_row0 = ((size_t)lc * prm.n_seqs_total + prm.seq_base + i) * c.n_q + (size_t)g * G;
  for (int e = tid; e < G * kHeadDim; e += kProfThreads)
    s_q[e / kHeadDim][e % kHeadDim] = __uint_as_float((uint32_t)prm.q[(q_row0 + e / kHeadDim) * kHeadDim + e % kHeadDim] << 16);
  if (tid == 0) {
    SeqParams cs = sp;
    if (prm.use_candidate) {
      cs.w_s = prm.cand.w_s; cs.d = prm.cand.d; cs.k_s = prm.cand.k_s; cs.w_o = prm.cand.w_o; cs.k_o = prm.cand.k_o;
    }
    Interval rr[6];
    s_ncand = retained_runs(cs, rr);
    for (int k = 0; k < s_ncand; ++k) s_cand[k] = rr[k];
  }
  __syncthreads();

  // ---- pass 1: scores ----
  const uint8_t* kp = reinterpret_cast<const uint8_t*>(c.k_pool);
  const int chunk = lane >> 1, half = lane & 1;
  for (int x = warp; x < len; x += kProfWarps) {
    bool is_dead = false;
    for (int k = 0; k < n_dead; ++k) is_dead |= (x >= dead[k].a && x < dead[k].b);
    const int page = is_dead ? -1 : tab[x >> plog];
    if (page < 0) {  // not resident
      if (lane < G) sc[(size_t)lane * prm.stride + x] = -INFINITY;
      continue;
    }
    const int slot = x & (p - 1);
    const int lchunk = chunk ^ (slot & 7);  // logical 16-byte chunk this lane's bytes belong to
    const uint2 kw = *reinterpret_cast<const uint2*>(kp + row_offset(c, layer, page, g, slot) + chunk * 16 + half * 8);
    const float k0 = bf_lo(kw.x), k1 = bf_hi(kw.x), k2 = bf_lo(kw.y), k3 = bf_hi(kw.y);
    const int d0 = lchunk * 8 + half * 4;
#pragma unroll
    for (int h = 0; h < kMaxGroup; ++h) {
      if (h < G) {
        const float4 qv = *reinterpret_cast<const float4*>(&s_q[h][d0]);
        float s = qv.x * k0 + qv.y * k1 + qv.z * k2 + qv.w * k3;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
        if (lane == 0) sc[(size_t)h * prm.stride + x] = s * prm.sm_scale;
      }
    }
  }
  __syncthreads();

  // positions are handled in contiguous per-thread chunks so that "ascending position" is thread order
  const int per = (len + kProfThreads - 1) / kProfThreads;
  const int x0 = min(len, tid * per), x1 = min(len, x0 + per);

  uint8_t* member = prm.member != nullptr ? prm.member + cta * (size_t)prm.stride : nullptr;
  if (member != nullptr)
    for (int x = x0; x < x1; ++x) member[x] = 0;  // each thread owns the positions [x0, x1) throughout

  for (int h = 0; h < G; ++h) {
    float* e = sc + (size_t)h * prm.stride;
    // ---- pass 2: softmax numerators, total, region masses, candidate coverage ----
    float mx = -INFINITY;
    for (int x = tid; x < len; x += kProfThreads) mx = fmaxf(mx, e[x]);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    __syncthreads();
    if (lane == 0) s_red[warp][0] = (double)mx;
    __syncthreads();
    float M = -INFINITY;
    for (int w = 0; w < kProfWarps; ++w) M = fmaxf(M, (float)s_red[w][0]);
    double acc[4] = {0.0, 0.0, 0.0, 0.0};  // prompt, speech, text, candidate
    int cnt[3] = {0, 0, 0};
    for (int x = x0; x < x1; ++x) {
      const float s = e[x];
      const float w = (s == -INFINITY) ? 0.f : __expf(s - M);
      e[x] = (s == -INFINITY) ? -1.f : w;  // -1 marks "not resident" from here on
      if (s == -INFINITY) continue;
      const int r = region_of(x, sp.P, sp.S, sp.M);
      acc[r] += (double)w;
      cnt[r] += 1;
      bool in = false;
      for (int k = 0; k < s_ncand; ++k) in |= (x >= s_cand[k].a && x < s_cand[k].b);
      if (in) acc[3] += (double)w;
    }
    double cd[4] = {(double)cnt[0], (double)cnt[1], (double)cnt[2], 0.0};
    block_sum4(acc, s_red);
    block_sum4(cd, s_red);
    const double L = acc[0] + acc[1] + acc[2];
    const double target = (double)prm.frac * L;

    // ---- pass 3: threshold weight by bisection on the bit pattern ----
    uint32_t tau = 0u;  // largest key with mass{e >= key} >= target (key 0 always qualifies)
    for (int bit = 30; bit >= 0; --bit) {
      const uint32_t trial = tau | (1u << bit);
      double m4[4] = {0.0, 0.0, 0.0, 0.0};
      for (int x = x0; x < x1; ++x) {
        const float w = e[x];
        if (w >= 0.f && __float_as_uint(w) >= trial) m4[0] += (double)w;
      }
      block_sum4(m4, s_red);
      if (m4[0] >= target) tau = trial;
    }
    // members above the threshold, per region, and the ties at it
    double gt[4] = {0.0, 0.0, 0.0, 0.0};  // counts per region of e > tau, and their mass
    int ties = 0;
    for (int x = x0; x < x1; ++x) {
      const float w = e[x];
      if (w < 0.f) continue;
      const uint32_t key = __float_as_uint(w);
      if (key > tau) {
        gt[region_of(x, sp.P, sp.S, sp.M)] += 1.0;
        gt[3] += (double)w;
        if (member != nullptr) member[x] = 1;
      } else if (key == tau) {
        ++ties;
      }
    }
    block_sum4(gt, s_red);
    const double w_tau = (double)__uint_as_float(tau);
    // ties needed, taken in ascending position: m = ceil((target - mass_gt) / w_tau), at least 1
    __syncthreads();
    s_scan[tid + 1] = ties;
    if (tid == 0) s_scan[0] = 0;
    __syncthreads();
    if (tid == 0)
      for (int k = 1; k <= kProfThreads; ++k) s_scan[k] += s_scan[k - 1];
    __syncthreads();
    const int total_ties = s_scan[kProfThreads];
    long long need = 1;
    if (w_tau > 0.0) {
      need = (long long)ceil((target - gt[3]) / w_tau);
      // guard the fp64 round trip: taking `need` ties must reach the target, need - 1 must not
      while (need > 1 && gt[3] + (double)(need - 1) * w_tau >= target) --need;
      while (need < total_ties && gt[3] + (double)need * w_tau < target) ++need;
    }
    if (need < 1) need = 1;
    if (need > total_ties) need = total_ties;
    double tk[4] = {0.0, 0.0, 0.0, 0.0};
    {
      int rank = s_scan[tid];
      for (int x = x0; x < x1 && rank < need; ++x) {
        const float w = e[x];
        if (w >= 0.f && __float_as_uint(w) == tau) {
          tk[region_of(x, sp.P, sp.S, sp.M)] += 1.0;
          if (member != nullptr) member[x] = 1;
          ++rank;
        }
      }
    }
    block_sum4(tk, s_red);
    if (tid == 0 && prm.out != nullptr) {
      murmur_profile_t r;
      r.n_prompt = (int32_t)cd[0];
      r.n_speech = (int32_t)cd[1];
      r.n_text = (int32_t)cd[2];
      r.n_resident = r.n_prompt + r.n_speech + r.n_text;
      r.k_prompt = (int32_t)(gt[0] + tk[0]);
      r.k_speech = (int32_t)(gt[1] + tk[1]);
      r.k_text = (int32_t)(gt[2] + tk[2]);
      r.k_mass = r.k_prompt + r.k_speech + r.k_text;
      r.coverage = (float)(acc[3] / L);
      r.mass_prompt = (float)(acc[0] / L);
      r.mass_speech = (float)(acc[1] / L);
      r.mass_text = (float)(acc[2] / L);
      prm.out[q_row0 + h] = r;
    }
    __syncthreads();
  }
}

}  // namespace

cudaError_t launch_attn_profile(const CacheView& c, const SeqList& list, int seq_base, int n_seqs_total, const void* q,
                                const SeqParams* candidate, float frac, void* out, float* scratch, long long stride,
                                int layer_begin, int layer_end, float sm_scale, uint8_t* member_mask, cudaStream_t st,
                                LaunchInfo* info) {
  ProfParams prm{};
  prm.member = member_mask;
  prm.q = reinterpret_cast<const uint16_t*>(q);
  prm.out = reinterpret_cast<murmur_profile_t*>(out);
  prm.scratch = scratch;
  prm.stride = stride;
  prm.seq_base = seq_base;
  prm.n_seqs_total = n_seqs_total;
  prm.layer_begin = layer_begin;
  prm.sm_scale = sm_scale;
  prm.frac = frac;
  prm.use_candidate = candidate != nullptr;
  if (candidate) prm.cand = *candidate;
  dim3 grid(c.n_kv, list.n, layer_end - layer_begin);
  attn_profile_kernel<<<grid, kProfThreads, 0, st>>>(c, list, prm);
  info->launches += 1;
  info->grid = (int)(grid.x * grid.y * grid.z);
  return cudaGetLastError();
}

// ---- the profile for callers that cannot provide scratch ------------------------------------------------------
// Same kernel, same arguments, but the per-head score rows go to murmur_profile_builtin_scratch instead of a
// buffer of the caller's.  Nothing is allocated here or anywhere below: one cudaGetDevice, on the first call per
// device one cudaGetSymbolAddress, and the launch.
//
// What the caller must know (repeated in murmur.h):
//   * the first call on a device looks the array's device address up; that look-up may load the module on the
//     device, so make this first call outside any stream capture;
//   * the array keeps whatever the previous call left in it.  The kernel needs no zeroed scratch: pass 1 writes
//     scratch[h][x] for every head h of the group and every x < len before pass 2 reads it, and nothing beyond
//     len is ever read, so there is nothing to clear;
//   * two calls in flight at once on one GPU (two streams, two handles, two threads) write the same rows and
//     corrupt each other's result.  Order them.
namespace {
constexpr int kMaxDevicesTracked = 64;
std::mutex g_builtin_mu;
float* g_builtin_ptr[kMaxDevicesTracked];  // device address of the array per device ordinal; null = not looked up yet
}  // namespace

cudaError_t launch_attn_profile_noalloc(const CacheView& c, const SeqList& list, int n_seqs_total, const void* q,
                                        const SeqParams* candidate, float frac, void* out, long long stride,
                                        size_t scratch_bytes_needed, int layer_begin, int layer_end, float sm_scale,
                                        cudaStream_t st, LaunchInfo* info) {
  if (scratch_bytes_needed > sizeof(murmur_profile_builtin_scratch)) return cudaErrorInvalidValue;  // API checks first
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kMaxDevicesTracked) return cudaErrorInvalidDevice;
  float* scratch = nullptr;
  {
    std::lock_guard<std::mutex> lk(g_builtin_mu);
    scratch = g_builtin_ptr[dev];
    if (scratch == nullptr) {
      void* p = nullptr;
      e = cudaGetSymbolAddress(&p, murmur_profile_builtin_scratch);  // address on the CURRENT device
      if (e != cudaSuccess) return e;
      if (p == nullptr) return cudaErrorInvalidSymbol;
      g_builtin_ptr[dev] = scratch = reinterpret_cast<float*>(p);
    }
  }
  return launch_attn_profile(c, list, 0, n_seqs_total, q, candidate, frac, out, scratch, stride, layer_begin,
                             layer_end, sm_scale, nullptr, st, info);
}

}  // namespace murmur
