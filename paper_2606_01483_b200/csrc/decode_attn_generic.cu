// murmur_decode_attn, generic variant: Eq. 1 over the retained set with plain
// FFMA, straight from global memory.  One CTA per (layer, sequence, KV head); each warp walks every
// 8th retained token through the run descriptors, keeps an fp32 online softmax for the G query
// heads of the group, and the warps' (m, l, o) partials are merged through shared memory with the
// log-sum-exp rule.  Works for every page size; it is the reference point the tensor-core kernel
// is measured against (and the path used for page_size < 16).
#include <cuda_bf16.h>

#include "device_state.cuh"

namespace murmur {
namespace {

constexpr int kGenWarps = 8;
constexpr int kGenThreads = kGenWarps * 32;

__device__ __forceinline__ float bf16_lo(uint32_t w) { return __uint_as_float(w << 16); }
__device__ __forceinline__ float bf16_hi(uint32_t w) { return __uint_as_float(w & 0xffff0000u); }

__global__ void __launch_bounds__(kGenThreads)
attn_generic_kernel(CacheView c, SeqList list, int seq_base, int n_seqs_total, const uint16_t* __restrict__ q,
                    uint16_t* __restrict__ out, float* __restrict__ lse, int layer_begin, float sm_scale) {
  __shared__ int s_run[kMaxRuns][3];
  __shared__ int s_run_off[kMaxRuns + 1];
  __shared__ float s_m[kGenWarps][kMaxGroup];
  __shared__ float s_l[kGenWarps][kMaxGroup];
  __shared__ float s_o[kGenWarps][kMaxGroup][kHeadDim];

  const int g = blockIdx.x;            // KV head
  const int i = blockIdx.y;            // index in this launch's sequence list
  const int lc = blockIdx.z;           // layer index inside the call
  const int layer = layer_begin + lc;
  const int id = list.ids[i];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int G = c.group;
  const SeqDev& sd = c.seqs[id];
  const int n_runs = sd.n_runs;
  if (threadIdx.x == 0) {
    int off = 0;
    for (int r = 0; r < n_runs; ++r) {
      s_run[r][0] = sd.runs[r][0];
      s_run[r][1] = sd.runs[r][1];
      s_run[r][2] = sd.runs[r][2];
      s_run_off[r] = off;
      off += sd.runs[r][1];
    }
    s_run_off[n_runs] = off;
  }
  __syncthreads();
  const int n_ret = s_run_off[n_runs];
  const int32_t* lpages = c.live_pages + (size_t)id * c.max_blocks;

  // this lane's 4 query dims of every head of the group
  const size_t q_row0 = ((size_t)lc * n_seqs_total + seq_base + i) * c.n_q + (size_t)g * G;
  float qv[kMaxGroup][4];
#pragma unroll
  for (int h = 0; h < kMaxGroup; ++h) {
    if (h < G) {
      const uint2 w = reinterpret_cast<const uint2*>(q + (q_row0 + h) * kHeadDim)[lane];
      qv[h][0] = bf16_lo(w.x); qv[h][1] = bf16_hi(w.x); qv[h][2] = bf16_lo(w.y); qv[h][3] = bf16_hi(w.y);
    } else {
      qv[h][0] = qv[h][1] = qv[h][2] = qv[h][3] = 0.f;
    }
  }
  float m[kMaxGroup], l[kMaxGroup], o[kMaxGroup][4];
#pragma unroll
  for (int h = 0; h < kMaxGroup; ++h) {
    m[h] = -INFINITY;
    l[h] = 0.f;
    o[h][0] = o[h][1] = o[h][2] = o[h][3] = 0.f;
  }

  const uint8_t* kp = reinterpret_cast<const uint8_t*>(c.k_pool);
  const uint8_t* vp = reinterpret_cast<const uint8_t*>(c.v_pool);
  const int chunk = lane >> 1, half = lane & 1;  // 16-byte chunk of the row and 8-byte half inside it
  for (int j = warp; j < n_ret; j += kGenWarps) {
    int r = 0;
    while (j >= s_run_off[r + 1]) ++r;
    const int x = s_run[r][0] + (j - s_run_off[r]);
    const int k = s_run[r][2] + ((x >> c.p_log2) - (s_run[r][0] >> c.p_log2));
    const int page = lpages[k];
    const int slot = x & (c.p - 1);
    const size_t off = row_offset(c, layer, page, g, slot) + (size_t)((chunk ^ (slot & 7)) * 16 + half * 8);
    const uint2 kw = *reinterpret_cast<const uint2*>(kp + off);
    const uint2 vw = *reinterpret_cast<const uint2*>(vp + off);
    const float k0 = bf16_lo(kw.x), k1 = bf16_hi(kw.x), k2 = bf16_lo(kw.y), k3 = bf16_hi(kw.y);
    const float v0 = bf16_lo(vw.x), v1 = bf16_hi(vw.x), v2 = bf16_lo(vw.y), v3 = bf16_hi(vw.y);
#pragma unroll
    for (int h = 0; h < kMaxGroup; ++h) {
      if (h < G) {
        float s = qv[h][0] * k0 + qv[h][1] * k1 + qv[h][2] * k2 + qv[h][3] * k3;
#pragma unroll
        for (int sh = 16; sh > 0; sh >>= 1) s += __shfl_xor_sync(0xffffffffu, s, sh);
        s *= sm_scale;
        const float mn = fmaxf(m[h], s);
        const float corr = __expf(m[h] - mn);
        const float pw = __expf(s - mn);
        l[h] = l[h] * corr + pw;
        o[h][0] = o[h][0] * corr + pw * v0;
        o[h][1] = o[h][1] * corr + pw * v1;
        o[h][2] = o[h][2] * corr + pw * v2;
        o[h][3] = o[h][3] * corr + pw * v3;
        m[h] = mn;
      }
    }
  }
#pragma unroll
  for (int h = 0; h < kMaxGroup; ++h) {
    if (lane == 0) {
      s_m[warp][h] = m[h];
      s_l[warp][h] = l[h];
    }
    s_o[warp][h][lane * 4 + 0] = o[h][0];
    s_o[warp][h][lane * 4 + 1] = o[h][1];
    s_o[warp][h][lane * 4 + 2] = o[h][2];
    s_o[warp][h][lane * 4 + 3] = o[h][3];
  }
  __syncthreads();
  // LSE merge of the 8 warp partials; thread -> (head, 4 dims)
  for (int e = threadIdx.x; e < G * kHeadDim; e += kGenThreads) {
    const int h = e / kHeadDim, d = e % kHeadDim;
    float M = -INFINITY;
#pragma unroll
    for (int w = 0; w < kGenWarps; ++w) M = fmaxf(M, s_m[w][h]);
    float L = 0.f, acc = 0.f;
#pragma unroll
    for (int w = 0; w < kGenWarps; ++w) {
      const float sc = (s_m[w][h] == -INFINITY) ? 0.f : __expf(s_m[w][h] - M);
      L += s_l[w][h] * sc;
      acc += s_o[w][h][d] * sc;
    }
    const size_t orow = q_row0 + h;
    out[orow * kHeadDim + d] = __bfloat16_as_ushort(__float2bfloat16_rn(acc / L));
    if (lse != nullptr && d == 0) lse[orow] = M + __logf(L);
  }
}

}  // namespace

cudaError_t launch_attn_generic(const CacheView& c, const SeqList& list, int seq_base, int n_seqs_total,
                                const void* q, void* out, float* lse, int layer_begin, int layer_end,
                                float sm_scale, cudaStream_t st, LaunchInfo* info) {
  dim3 grid(c.n_kv, list.n, layer_end - layer_begin);
  attn_generic_kernel<<<grid, kGenThreads, 0, st>>>(c, list, seq_base, n_seqs_total,
                                                    reinterpret_cast<const uint16_t*>(q),
                                                    reinterpret_cast<uint16_t*>(out), lse, layer_begin, sm_scale);
  info->launches += 1;
  info->grid = (int)(grid.x * grid.y * grid.z);
  info->smem = 0;
  return cudaGetLastError();
}

}  // namespace murmur
