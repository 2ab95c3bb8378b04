// murmur_decode_attn_indexed on the tensor cores: Eq. 1 of the 7 query heads of a GQA
// group over the rows of ONE slab (layer, KV head) of a sequence in indexed mode (general index-set
// eviction).
//
// A slab is dense: row j is slot j mod p of the sequence's block j div p, for j < len(layer, head), and
// every (layer, head) has its own length - so, unlike the positional path, there is no tile list shared by
// all layers and heads of a sequence, and the work item is simply (layer, sequence, KV head): one CTA
// streams that slab once.  HBM-bound like the positional decode kernel, and built from the same parts:
//   warp 8       producer: 1-D bulk copies (TMA engine) of whole (page, head) chunks - p x 256 contiguous
//                bytes, pre-swizzled in the pool for ldmatrix - into a 4-stage ring of 64-row K and V tiles,
//                completion counted in bytes on mbarriers, L2::evict_first;
//   warps 0-7    two groups of four: a group takes every second tile, a warp 16 of its 64 rows:
//                S^T[16 x 8] = K Q^T and O^T[128 x 8] += V^T P^T with mma.sync.m16n8k16 (tokens are M, the
//                group's heads N = 8), fp32 online softmax in the exp2 domain;
//   end of slab  the eight (m, l, O^T) states are merged in the MMA fragment layout through shared memory.
// Pages must hold a multiple of 16 rows (p = 16, 32, 64); other page sizes keep the FFMA kernel.
#include <cuda_bf16.h>

#include "device_state.cuh"
#include "ptx_utils.cuh"

namespace murmur {
namespace {

constexpr int kXStages = 4;
constexpr int kXConsumers = 8;                      // consumer warps (two groups of four)
constexpr int kXThreads = (kXConsumers + 1) * 32;
constexpr int kXTileBytes = kTileRows * kRowBytes;  // 16 KB: 64 rows of K (or V) of one head

struct __align__(128) XSmem {
  uint8_t kv[kXStages][2][kXTileBytes];             // [stage][K | V]
  float frag[kXConsumers][kPartialFloats];          // (O^T, m, l) of every consumer warp, fragment layout
  unsigned long long full_k[kXStages], full_v[kXStages], empty[kXStages];
};

__global__ void __launch_bounds__(kXThreads, 1)
indexed_attn_mma_kernel(const __grid_constant__ CacheView c, const __grid_constant__ IdxView ix,
                        const __grid_constant__ SeqList list, const uint16_t* __restrict__ q, uint16_t* __restrict__ out,
                        float* __restrict__ lse, float sm_scale) {
  extern __shared__ uint8_t xsmem_raw[];
  XSmem& s = *reinterpret_cast<XSmem*>(xsmem_raw + ((128u - (smem_u32(xsmem_raw) & 127u)) & 127u));
  const int g = blockIdx.x, i = blockIdx.y, layer = blockIdx.z;
  const int id = list.ids[i];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int G = c.group, p = c.p, plog = c.p_log2;
  const int n = ix.len[(size_t)id * c.n_layers * c.n_kv + layer * c.n_kv + g];   // rows of this slab
  const int n_tiles = (n + kTileRows - 1) / kTileRows;
  const size_t q_row0 = ((size_t)layer * list.n + i) * c.n_q + (size_t)g * G;

  if (threadIdx.x == 0) {
    for (int st = 0; st < kXStages; ++st) {
      mbar_init(&s.full_k[st], 1);
      mbar_init(&s.full_v[st], 1);
      mbar_init(&s.empty[st], 4);   // the four warps of the group that consumed the tile
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  if (warp == kXConsumers) {
    // ===================================== producer =====================================
    if (lane == 0) {
      const int32_t* tab = c.block_table + (size_t)id * c.max_blocks;
      const uint8_t* kp = reinterpret_cast<const uint8_t*>(c.k_pool);
      const uint8_t* vp = reinterpret_cast<const uint8_t*>(c.v_pool);
      const unsigned long long pol = l2_policy_evict_first();
      const int ppt = kTileRows >> plog;  // pages per tile
      const uint32_t chunk = (uint32_t)p * kRowBytes;
      for (int t = 0; t < n_tiles; ++t) {
        const int st = t % kXStages;
        mbar_wait(&s.empty[st], (uint32_t)((t / kXStages) & 1) ^ 1u);
        const int rows = min(kTileRows, n - t * kTileRows);
        const int pages = (rows + p - 1) >> plog;   // whole pages; rows past n inside the last one are masked
        mbar_expect_tx(&s.full_k[st], (uint32_t)pages * chunk);
        mbar_expect_tx(&s.full_v[st], (uint32_t)pages * chunk);
        for (int pg = 0; pg < pages; ++pg) {
          const size_t off = row_offset(c, layer, tab[t * ppt + pg], g, 0);
          bulk_g2s_hint(&s.kv[st][0][(size_t)pg * chunk], kp + off, chunk, &s.full_k[st], pol);
        }
        for (int pg = 0; pg < pages; ++pg) {
          const size_t off = row_offset(c, layer, tab[t * ppt + pg], g, 0);
          bulk_g2s_hint(&s.kv[st][1][(size_t)pg * chunk], vp + off, chunk, &s.full_v[st], pol);
        }
      }
    }
    return;
  }

  // ===================================== consumer warps =====================================
  const float c2 = sm_scale * 1.4426950408889634f;  // scores are kept raw; exp2((s - m) * c2)
  const int w4 = warp & 3, grp = warp >> 2;
  const int lrow = lane >> 2;         // row inside an 8-row group / head index of B fragments
  const int lcol = (lane & 3) * 2;    // first of the two heads (or tokens) this lane owns
  // ldmatrix lane addressing (row inside the 16-row group, 16-byte chunk select, swizzle key)
  const int lm_row = ((lane >> 3) & 1) * 8 + (lane & 7);  // K (non-transposed): matrices 0..3 =
  const int lm_chk = lane >> 4;                           //   (rows 0-7, c), (8-15, c), (0-7, c+1), (8-15, c+1)
  const int lv_row = (lane >> 4) * 8 + (lane & 7);        // V (transposed): (rows 0-7, c), (0-7, c+1),
  const int lv_chk = (lane >> 3) & 1;                     //   (8-15, c), (8-15, c+1)
  const int key = lane & 7;                               // tiles start at slot 0 of a page: row & 7 == slot & 7
  const int slice0 = w4 * 16;                             // first row of this warp's slice
  const uint32_t k_off = (uint32_t)(slice0 + lm_row) * kRowBytes;
  const uint32_t v_off = (uint32_t)(slice0 + lv_row) * kRowBytes;

  // query fragments (B operand of S^T = K Q^T): head lrow, d = 16 ks + lcol (+1) and + 8; heads >= G are zero
  uint32_t qf[8][2];
  {
    const uint16_t* qs = q + (q_row0 + (size_t)min(lrow, G - 1)) * kHeadDim + lcol;
#pragma unroll
    for (int ks = 0; ks < 8; ++ks) {
      const uint32_t a = *reinterpret_cast<const uint32_t*>(qs + ks * 16);
      const uint32_t b = *reinterpret_cast<const uint32_t*>(qs + ks * 16 + 8);
      qf[ks][0] = lrow < G ? a : 0u;
      qf[ks][1] = lrow < G ? b : 0u;
    }
  }
  float m0 = -INFINITY, m1 = -INFINITY, l0 = 0.f, l1 = 0.f;
  float o[8][4];
#pragma unroll
  for (int dt = 0; dt < 8; ++dt) o[dt][0] = o[dt][1] = o[dt][2] = o[dt][3] = 0.f;

  for (int t = grp; t < n_tiles; t += 2) {
    const int st = t % kXStages;
    const uint32_t ph = (uint32_t)(t / kXStages) & 1u;
    const int re = min(kTileRows, n - t * kTileRows);   // valid rows of the tile: [0, re)
    const bool act = slice0 < re;                       // warp-uniform: the slice holds a valid row
    uint32_t pb0 = 0u, pb1 = 0u;
    mbar_wait(&s.full_k[st], ph);
    if (act) {
      // ---- S^T[16 x 8] = K Q^T, two independent accumulator chains ----
      const uint32_t rowaddr = smem_u32(&s.kv[st][0][0]) + k_off;
      float sa[4] = {0.f, 0.f, 0.f, 0.f}, sb[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
      for (int ks = 0; ks < 8; ks += 2) {
        uint32_t a[4], b[4];
        ldsm_x4(a, rowaddr + (uint32_t)(((2 * ks + lm_chk) ^ key) << 4));
        ldsm_x4(b, rowaddr + (uint32_t)(((2 * ks + 2 + lm_chk) ^ key) << 4));
        mma_bf16(sa, a, qf[ks][0], qf[ks][1]);
        mma_bf16(sb, b, qf[ks + 1][0], qf[ks + 1][1]);
      }
      float s0 = sa[0] + sb[0], s1 = sa[1] + sb[1], s2 = sa[2] + sb[2], s3 = sa[3] + sb[3];
      const int r0 = slice0 + lrow, r1 = r0 + 8;
      if (r0 >= re) s0 = s1 = -INFINITY;
      if (r1 >= re) s2 = s3 = -INFINITY;
      float mx0 = fmaxf(s0, s2), mx1 = fmaxf(s1, s3);
#pragma unroll
      for (int sh = 4; sh <= 16; sh <<= 1) {
        mx0 = fmaxf(mx0, __shfl_xor_sync(0xffffffffu, mx0, sh));
        mx1 = fmaxf(mx1, __shfl_xor_sync(0xffffffffu, mx1, sh));
      }
      const float mn0 = fmaxf(m0, mx0), mn1 = fmaxf(m1, mx1);  // finite: the slice has a valid row
      if (__any_sync(0xffffffffu, (mn0 != m0) || (mn1 != m1))) {
        const float cr0 = ex2((m0 - mn0) * c2), cr1 = ex2((m1 - mn1) * c2);
        m0 = mn0;
        m1 = mn1;
        l0 *= cr0;
        l1 *= cr1;
#pragma unroll
        for (int dt = 0; dt < 8; ++dt) {
          o[dt][0] *= cr0; o[dt][1] *= cr1; o[dt][2] *= cr0; o[dt][3] *= cr1;
        }
      }
      // ---- P^T fragment: exp2, bf16, transpose into the B-operand layout ----
      const float ms0 = m0 * c2, ms1 = m1 * c2;
      const float p0 = ex2(s0 * c2 - ms0), p1 = ex2(s1 * c2 - ms1);
      const float p2 = ex2(s2 * c2 - ms0), p3 = ex2(s3 * c2 - ms1);
      l0 += p0 + p2;
      l1 += p1 + p3;
      pb0 = movmatrix_t(pack_bf16(p0, p1));
      pb1 = movmatrix_t(pack_bf16(p2, p3));
    }
    // ---- O^T[128 x 8] += V^T P^T over this warp's 16 rows ----
    mbar_wait(&s.full_v[st], ph);
    if (act) {
      const uint32_t rowaddr = smem_u32(&s.kv[st][1][0]) + v_off;
      uint32_t mk01 = 0xffffffffu, mk23 = 0xffffffffu;
      if (slice0 + 16 > re) {  // rows at or past re hold whatever the pool (or an older tile) held: zero them in the A fragment
        const int t0 = slice0 + lcol;
        mk01 = (t0 < re ? 0x0000ffffu : 0u) | (t0 + 1 < re ? 0xffff0000u : 0u);
        mk23 = (t0 + 8 < re ? 0x0000ffffu : 0u) | (t0 + 9 < re ? 0xffff0000u : 0u);
      }
#pragma unroll
      for (int dt = 0; dt < 8; ++dt) {
        uint32_t a[4];
        ldsm_x4_t(a, rowaddr + (uint32_t)(((2 * dt + lv_chk) ^ key) << 4));
        a[0] &= mk01; a[1] &= mk01; a[2] &= mk23; a[3] &= mk23;
        mma_bf16(o[dt], a, pb0, pb1);
      }
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(&s.empty[st]);
  }

  // ---- merge of the eight warps' states, lane for lane in the fragment layout; warp 0 writes the output ----
  {
    float* fs = s.frag[warp];
#pragma unroll
    for (int dt = 0; dt < 8; ++dt) {
#pragma unroll
      for (int e = 0; e < 4; ++e) fs[(dt * 4 + e) * 32 + lane] = o[dt][e];
    }
    fs[32 * 32 + lane] = m0;
    fs[33 * 32 + lane] = m1;
    fs[34 * 32 + lane] = l0;
    fs[35 * 32 + lane] = l1;
  }
  asm volatile("bar.sync 1, %0;" ::"n"(kXConsumers * 32) : "memory");
  if (warp != 0) return;
  for (int wv = 1; wv < kXConsumers; ++wv) {
    const float* fs = s.frag[wv];
    const float mo0 = fs[32 * 32 + lane], mo1 = fs[33 * 32 + lane];
    const float mn0 = fmaxf(m0, mo0), mn1 = fmaxf(m1, mo1);
    const float fa0 = (m0 == -INFINITY) ? 0.f : ex2((m0 - mn0) * c2);
    const float fa1 = (m1 == -INFINITY) ? 0.f : ex2((m1 - mn1) * c2);
    const float fb0 = (mo0 == -INFINITY) ? 0.f : ex2((mo0 - mn0) * c2);
    const float fb1 = (mo1 == -INFINITY) ? 0.f : ex2((mo1 - mn1) * c2);
    l0 = l0 * fa0 + fs[34 * 32 + lane] * fb0;
    l1 = l1 * fa1 + fs[35 * 32 + lane] * fb1;
#pragma unroll
    for (int dt = 0; dt < 8; ++dt) {
      o[dt][0] = o[dt][0] * fa0 + fs[(dt * 4 + 0) * 32 + lane] * fb0;
      o[dt][1] = o[dt][1] * fa1 + fs[(dt * 4 + 1) * 32 + lane] * fb1;
      o[dt][2] = o[dt][2] * fa0 + fs[(dt * 4 + 2) * 32 + lane] * fb0;
      o[dt][3] = o[dt][3] * fa1 + fs[(dt * 4 + 3) * 32 + lane] * fb1;
    }
    m0 = mn0;
    m1 = mn1;
  }
  // lane (lrow, lcol) holds O^T[d][head] for d = 16 dt + lrow (+ 8), head = lcol (+ 1); l is still split over lrow
  float t0 = l0, t1 = l1;
#pragma unroll
  for (int sh = 4; sh <= 16; sh <<= 1) {
    t0 += __shfl_xor_sync(0xffffffffu, t0, sh);
    t1 += __shfl_xor_sync(0xffffffffu, t1, sh);
  }
  const float i0 = 1.f / t0, i1 = 1.f / t1;
  uint16_t* o0 = out + (q_row0 + lcol) * kHeadDim;
  uint16_t* o1 = o0 + kHeadDim;
#pragma unroll
  for (int dt = 0; dt < 8; ++dt) {
    const int d = dt * 16 + lrow;
    if (lcol < G) {
      o0[d] = __bfloat16_as_ushort(__float2bfloat16_rn(o[dt][0] * i0));
      o0[d + 8] = __bfloat16_as_ushort(__float2bfloat16_rn(o[dt][2] * i0));
    }
    if (lcol + 1 < G) {
      o1[d] = __bfloat16_as_ushort(__float2bfloat16_rn(o[dt][1] * i1));
      o1[d + 8] = __bfloat16_as_ushort(__float2bfloat16_rn(o[dt][3] * i1));
    }
  }
  if (lse != nullptr && lrow == 0) {
    if (lcol < G) lse[q_row0 + lcol] = m0 * sm_scale + __logf(t0);
    if (lcol + 1 < G) lse[q_row0 + lcol + 1] = m1 * sm_scale + __logf(t1);
  }
}

}  // namespace

cudaError_t launch_indexed_attn_mma(const CacheView& c, const IdxView& ix, const SeqList& list, const void* q, void* out,
                                    float* lse, float sm_scale, cudaStream_t st, LaunchInfo* info) {
  const int smem = (int)sizeof(XSmem) + 128;
  cudaError_t ea = opt_in_smem_once(kSmemIndexed, reinterpret_cast<const void*>(indexed_attn_mma_kernel), smem);
  if (ea != cudaSuccess) return ea;
  dim3 grid(c.n_kv, list.n, c.n_layers);
  indexed_attn_mma_kernel<<<grid, kXThreads, smem, st>>>(c, ix, list, reinterpret_cast<const uint16_t*>(q),
                                                         reinterpret_cast<uint16_t*>(out), lse, sm_scale);
  info->launches += 1;
  info->grid = (int)(grid.x * grid.y * grid.z);
  info->smem = smem;
  return cudaGetLastError();
}

}  // namespace murmur
