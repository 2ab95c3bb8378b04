// murmur_prefill_attn: causal self-attention of a sequence's prefill tokens over the paged cache.
//
// PAPER.md:95 (chunks are submitted to the engine as a batch; the engine first runs prompt + speech
// tokens through the model) and PAPER.md:77 (prefill = what is left of model time after the 95.3 %
// of decoding).  Position x attends, by Eq. 1, to the cache positions y <= x.
// The K/V rows are read from the pools murmur_kv_append filled (pre-swizzled rows: a 1-D bulk copy
// of a page lands conflict-free for ldmatrix), so prefill and decode share one cache layout.
//
// One CTA per (64-query tile, query head, layer), heaviest tiles first.  4 consumer warps own 16
// query rows each; 1 producer warp streams 64-key K/V tiles through a 3-stage ring with
// cp.async.bulk.  Per tile and warp: S[16 x 64] = Q K^T (mma.sync m16n8k16 bf16, Q fragments kept in
// registers), causal mask on the diagonal tile, fp32 online softmax (exp2 form), P re-used from
// the accumulator layout as the A operand of O[16 x 128] += P V (V through ldmatrix.trans).
// FIRST CORRECT PATH: mma.sync, not yet tcgen05/TMEM - a dense contraction of this shape
// (M = 64 queries x 7 heads per KV head) is where tcgen05 belongs; see DESIGN.md section 9.
#include <cuda_bf16.h>

#include "device_state.cuh"
#include "ptx_utils.cuh"

namespace murmur {
namespace {

constexpr int kPfStages = 3;
constexpr int kPfConsumerWarps = 4;
constexpr int kPfThreads = (kPfConsumerWarps + 1) * 32;
constexpr int kPfTile = 64;                          // queries per CTA and keys per tile
constexpr int kPfTileBytes = kPfTile * kRowBytes;    // 16 KB

struct __align__(128) PfSmem {
  uint8_t kv[kPfStages][2][kPfTileBytes];
  uint8_t q[kPfTileBytes];
  unsigned long long full[kPfStages], empty[kPfStages];
};

struct PfParams {
  const uint16_t* q;   // [layers][n_tok][n_q][128]
  uint16_t* out;       // same
  float* lse;          // [layers][n_tok][n_q] or null
  int seq, pos_begin, n_tok, layer_begin;
  float sm_scale;
};

__global__ void __launch_bounds__(kPfThreads, 2)
prefill_attn_kernel(const __grid_constant__ CacheView c, const __grid_constant__ PfParams prm) {
  extern __shared__ __align__(128) uint8_t smem_raw[];
  PfSmem& s = *reinterpret_cast<PfSmem*>(smem_raw);
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int n_qt = (prm.n_tok + kPfTile - 1) / kPfTile;
  const int qt = n_qt - 1 - (int)blockIdx.x;  // heaviest (latest) query tiles first
  const int h = blockIdx.y, lc = blockIdx.z;
  const int layer = prm.layer_begin + lc;
  const int kvh = h / c.group;
  const int p = c.p, plog = c.p_log2;
  const int x0 = prm.pos_begin + qt * kPfTile;                      // first query position of the tile
  const int x_last = min(prm.pos_begin + prm.n_tok, x0 + kPfTile) - 1;  // last valid one
  const int n_kt = (x_last >> 6) + 1;                               // key tiles 0 .. n_kt-1 (64-aligned)

  if (tid == 0) {
    for (int i = 0; i < kPfStages; ++i) {
      mbar_init(&s.full[i], 1);
      mbar_init(&s.empty[i], kPfConsumerWarps);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  if (warp == kPfConsumerWarps) {
    // ---------------- producer: K and V tiles of 64 positions = 64/p pages ----------------
    if (lane == 0) {
      const int32_t* tab = c.block_table + (size_t)prm.seq * c.max_blocks;
      const uint8_t* kpool = reinterpret_cast<const uint8_t*>(c.k_pool);
      const uint8_t* vpool = reinterpret_cast<const uint8_t*>(c.v_pool);
      const int ppt = kPfTile >> plog;
      for (int j = 0; j < n_kt; ++j) {
        const int st = j % kPfStages;
        const uint32_t ph = (j / kPfStages) & 1u;
        mbar_wait(&s.empty[st], ph ^ 1u);
        const int rows = min(kPfTile, x_last + 1 - j * kPfTile);  // keys beyond x_last are never needed
        mbar_expect_tx(&s.full[st], 2u * (uint32_t)rows * kRowBytes);
        for (int pg = 0; pg < ppt; ++pg) {
          const int r0 = pg * p;
          if (r0 >= rows) break;
          const int nr = min(p, rows - r0);
          const int page = tab[j * ppt + pg];
          const size_t off = row_offset(c, layer, page, kvh, 0);
          bulk_g2s(&s.kv[st][0][r0 * kRowBytes], kpool + off, (uint32_t)nr * kRowBytes, &s.full[st]);
          bulk_g2s(&s.kv[st][1][r0 * kRowBytes], vpool + off, (uint32_t)nr * kRowBytes, &s.full[st]);
        }
      }
    }
    return;
  }

  // ---------------- consumers ----------------
  // Q tile -> shared memory, swizzled like the pool rows (chunk c of row r at c ^ (r & 7))
  for (int e = tid; e < kPfTile * 16; e += kPfConsumerWarps * 32) {
    const int r = e >> 4, ch = e & 15;
    const int x = x0 + r;
    uint4 val = make_uint4(0u, 0u, 0u, 0u);
    if (x <= x_last) {
      const size_t row = ((size_t)lc * prm.n_tok + (x - prm.pos_begin)) * c.n_q + h;
      val = reinterpret_cast<const uint4*>(prm.q + row * kHeadDim)[ch];
    }
    *reinterpret_cast<uint4*>(&s.q[r * kRowBytes + ((ch ^ (r & 7)) << 4)]) = val;
  }
  asm volatile("bar.sync 1, %0;" ::"n"(kPfConsumerWarps * 32) : "memory");

  const int key = lane & 7;
  // A-operand (m16 x k16) addressing: matrices (rows 0-7, c), (8-15, c), (0-7, c+1), (8-15, c+1)
  const int la_row = ((lane >> 3) & 1) * 8 + (lane & 7), la_chk = lane >> 4;
  uint32_t qa[8][4];
  {
    const uint32_t base = smem_u32(&s.q[0]) + (uint32_t)(warp * 16 + la_row) * kRowBytes;
#pragma unroll
    for (int ks = 0; ks < 8; ++ks) ldsm_x4(qa[ks], base + (uint32_t)(((2 * ks + la_chk) ^ key) << 4));
  }
  const float c2 = prm.sm_scale * 1.4426950408889634f;
  const int xr0 = x0 + warp * 16 + (lane >> 2), xr1 = xr0 + 8;  // this thread's two query positions
  float m0 = -INFINITY, m1 = -INFINITY, l0 = 0.f, l1 = 0.f;
  float o[16][4];
#pragma unroll
  for (int dt = 0; dt < 16; ++dt) o[dt][0] = o[dt][1] = o[dt][2] = o[dt][3] = 0.f;

  // B-operand addressing.  K (non-transposed, n = keys): matrices = 16-byte chunks 4q .. 4q+3 of
  // keys nt*8 + (lane & 7).  V (transposed, n = d): (keys 0-7, c), (8-15, c), (0-7, c+1), (8-15, c+1).
  const int lk_chk = lane >> 3;
  const int lv_row = ((lane >> 3) & 1) * 8 + (lane & 7), lv_chk = lane >> 4;

  for (int j = 0; j < n_kt; ++j) {
    const int st = j % kPfStages;
    const uint32_t ph = (j / kPfStages) & 1u;
    const int y0 = j * kPfTile;
    // a warp whose 16 queries all precede this key tile has nothing to do in it
    const bool warp_active = y0 <= x0 + warp * 16 + 15;
    mbar_wait(&s.full[st], ph);
    if (warp_active) {
      float sc[8][4];
      const uint32_t kbase = smem_u32(&s.kv[st][0][0]);
#pragma unroll
      for (int nt = 0; nt < 8; ++nt) {
        sc[nt][0] = sc[nt][1] = sc[nt][2] = sc[nt][3] = 0.f;
        const uint32_t rowaddr = kbase + (uint32_t)(nt * 8 + (lane & 7)) * kRowBytes;
#pragma unroll
        for (int qd = 0; qd < 4; ++qd) {
          uint32_t b[4];
          ldsm_x4(b, rowaddr + (uint32_t)(((4 * qd + lk_chk) ^ key) << 4));
          mma_bf16(sc[nt], qa[2 * qd], b[0], b[1]);
          mma_bf16(sc[nt], qa[2 * qd + 1], b[2], b[3]);
        }
      }
      // causal mask (also hides the rows of a partial last tile that were never copied)
      if (y0 + kPfTile - 1 > x0 + warp * 16) {
#pragma unroll
        for (int nt = 0; nt < 8; ++nt) {
          const int y = y0 + nt * 8 + (lane & 3) * 2;
          if (y > xr0) sc[nt][0] = -INFINITY;
          if (y + 1 > xr0) sc[nt][1] = -INFINITY;
          if (y > xr1) sc[nt][2] = -INFINITY;
          if (y + 1 > xr1) sc[nt][3] = -INFINITY;
        }
      }
      float mx0 = -INFINITY, mx1 = -INFINITY;
#pragma unroll
      for (int nt = 0; nt < 8; ++nt) {
        mx0 = fmaxf(mx0, fmaxf(sc[nt][0], sc[nt][1]));
        mx1 = fmaxf(mx1, fmaxf(sc[nt][2], sc[nt][3]));
      }
      mx0 = fmaxf(mx0, __shfl_xor_sync(0xffffffffu, mx0, 1));
      mx0 = fmaxf(mx0, __shfl_xor_sync(0xffffffffu, mx0, 2));
      mx1 = fmaxf(mx1, __shfl_xor_sync(0xffffffffu, mx1, 1));
      mx1 = fmaxf(mx1, __shfl_xor_sync(0xffffffffu, mx1, 2));
      // key 0 <= every query position: after the first tile the running max is finite
      const float mn0 = fmaxf(m0, mx0), mn1 = fmaxf(m1, mx1);
      const float cr0 = (m0 == -INFINITY) ? 0.f : ex2((m0 - mn0) * c2);
      const float cr1 = (m1 == -INFINITY) ? 0.f : ex2((m1 - mn1) * c2);
      m0 = mn0;
      m1 = mn1;
      l0 *= cr0;
      l1 *= cr1;
#pragma unroll
      for (int dt = 0; dt < 16; ++dt) {
        o[dt][0] *= cr0; o[dt][1] *= cr0; o[dt][2] *= cr1; o[dt][3] *= cr1;
      }
      const float ms0 = (m0 == -INFINITY) ? 0.f : m0 * c2, ms1 = (m1 == -INFINITY) ? 0.f : m1 * c2;
      uint32_t pa[4][4];  // P as A operand: k-step kk covers keys 16 kk .. 16 kk + 15 = n-tiles 2kk, 2kk+1
#pragma unroll
      for (int nt = 0; nt < 8; ++nt) {
        const float p0 = ex2(sc[nt][0] * c2 - ms0), p1 = ex2(sc[nt][1] * c2 - ms0);
        const float p2 = ex2(sc[nt][2] * c2 - ms1), p3 = ex2(sc[nt][3] * c2 - ms1);
        l0 += p0 + p1;
        l1 += p2 + p3;
        pa[nt >> 1][(nt & 1) * 2 + 0] = pack_bf16(p0, p1);
        pa[nt >> 1][(nt & 1) * 2 + 1] = pack_bf16(p2, p3);
      }
      const uint32_t vbase = smem_u32(&s.kv[st][1][0]);
      const int rows = min(kPfTile, x_last + 1 - y0);  // valid key rows of this tile
#pragma unroll
      for (int kk = 0; kk < 4; ++kk) {
        if (kk * 16 < rows) {  // rows beyond were never copied (their P is 0, but stale bits could be NaN)
          const uint32_t rowaddr = vbase + (uint32_t)(kk * 16 + lv_row) * kRowBytes;
#pragma unroll
          for (int dp = 0; dp < 8; ++dp) {
            uint32_t b[4];
            ldsm_x4_t(b, rowaddr + (uint32_t)(((2 * dp + lv_chk) ^ key) << 4));
            if (kk * 16 + 16 > rows) {  // partially valid 16-key group: zero the stale keys' V
              const int k0 = kk * 16 + (lane & 3) * 2;
              const uint32_t mlo = ((k0 < rows) ? 0x0000ffffu : 0u) | ((k0 + 1 < rows) ? 0xffff0000u : 0u);
              const uint32_t mhi = ((k0 + 8 < rows) ? 0x0000ffffu : 0u) | ((k0 + 9 < rows) ? 0xffff0000u : 0u);
              b[0] &= mlo; b[1] &= mhi; b[2] &= mlo; b[3] &= mhi;
            }
            mma_bf16(o[2 * dp], pa[kk], b[0], b[1]);
            mma_bf16(o[2 * dp + 1], pa[kk], b[2], b[3]);
          }
        }
      }
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(&s.empty[st]);
  }

  // ---------------- epilogue ----------------
  l0 += __shfl_xor_sync(0xffffffffu, l0, 1);
  l0 += __shfl_xor_sync(0xffffffffu, l0, 2);
  l1 += __shfl_xor_sync(0xffffffffu, l1, 1);
  l1 += __shfl_xor_sync(0xffffffffu, l1, 2);
  const float i0 = 1.f / l0, i1 = 1.f / l1;
  const int dcol = (lane & 3) * 2;
  if (xr0 <= x_last) {
    const size_t row = ((size_t)lc * prm.n_tok + (xr0 - prm.pos_begin)) * c.n_q + h;
#pragma unroll
    for (int dt = 0; dt < 16; ++dt)
      *reinterpret_cast<uint32_t*>(prm.out + row * kHeadDim + dt * 8 + dcol) = pack_bf16(o[dt][0] * i0, o[dt][1] * i0);
    if (prm.lse != nullptr && (lane & 3) == 0) prm.lse[row] = m0 * prm.sm_scale + __logf(l0);
  }
  if (xr1 <= x_last) {
    const size_t row = ((size_t)lc * prm.n_tok + (xr1 - prm.pos_begin)) * c.n_q + h;
#pragma unroll
    for (int dt = 0; dt < 16; ++dt)
      *reinterpret_cast<uint32_t*>(prm.out + row * kHeadDim + dt * 8 + dcol) = pack_bf16(o[dt][2] * i1, o[dt][3] * i1);
    if (prm.lse != nullptr && (lane & 3) == 0) prm.lse[row] = m1 * prm.sm_scale + __logf(l1);
  }
}

}  // namespace

cudaError_t launch_prefill_attn(const CacheView& c, int seq, int pos_begin, int n_tok, const void* q, void* out,
                                float* lse, int layer_begin, int layer_end, float sm_scale, cudaStream_t st,
                                LaunchInfo* info) {
  const int smem = (int)sizeof(PfSmem);
  cudaError_t ea = opt_in_smem_once(kSmemPrefill, reinterpret_cast<const void*>(prefill_attn_kernel), smem);
  if (ea != cudaSuccess) return ea;
  PfParams prm{};
  prm.q = reinterpret_cast<const uint16_t*>(q);
  prm.out = reinterpret_cast<uint16_t*>(out);
  prm.lse = lse;
  prm.seq = seq;
  prm.pos_begin = pos_begin;
  prm.n_tok = n_tok;
  prm.layer_begin = layer_begin;
  prm.sm_scale = sm_scale;
  dim3 grid((n_tok + kPfTile - 1) / kPfTile, c.n_q, layer_end - layer_begin);
  prefill_attn_kernel<<<grid, kPfThreads, smem, st>>>(c, prm);
  info->launches += 1;
  info->grid = (int)(grid.x * grid.y * grid.z);
  info->smem = smem;
  return cudaGetLastError();
}

}  // namespace murmur
