// murmur_decode_attn, tensor-core split-K variant for sm_100a.
//
// Eq. 1 for one query token per sequence over the retained set, all layers in
// ONE persistent launch (the path moves only ~20 MB per layer, so per-layer launches could never
// reach the HBM roofline - DESIGN.md "Kernels").
//
// Work decomposition
//   item  = (layer, sequence, KV head): G query heads (<= 8) share every K/V row.
//   tile  = <= 64 consecutive retained rows of one run (64/p consecutive live pages), built by
//           murmur_kv_evict; identical for all layers and heads of a sequence.
//   The flattened tile list (layer, seq, head, tile) is cut into `grid` equal contiguous ranges,
//   one per CTA (split-K across the retained length whenever a cut falls inside an item).
// Per CTA: 1 producer warp + 6 consumer warps, a 6-stage ring of (K tile, V tile) buffers
//   (tile n lives in stage n % 6 and is consumed by warp n % 6, so each stage has one owner).
//   producer : one lane per tile issues 1-D bulk copies (cp.async.bulk, TMA engine) of each
//              page's contiguous row range straight into the stage buffer; rows are stored
//              pre-swizzled in HBM, so the copy needs no tensor map and ldmatrix is
//              conflict-free.  Bytes copied = retained rows exactly.
//   consumer : warp w takes every 6th tile.  S^T[64 tok x 8 heads] = K Q^T with mma.sync
//              m16n8k16 bf16 (tokens are M, the padded head group is N: 7/8 useful), fp32
//              online softmax in exp2 form, P^T moved to the B-operand layout with movmatrix,
//              O^T[128 d x 8 heads] += V^T P^T with ldmatrix.trans.
//   merge    : the six warps' (m, l, O) are merged through shared memory; an item that spans
//              several CTAs is finished by the LAST contributor (arrival counter): partials go
//              to a workspace slot, the last one merges them by the log-sum-exp rule.
#include <cuda_bf16.h>

#include "device_state.cuh"

namespace murmur {
namespace {

constexpr int kStages = 6;
constexpr int kSliceWarps = 4;   // the four 16-row slices of a 64-row tile, one warp each
constexpr int kGroups = 2;       // warp groups; group g consumes tiles n with n % kGroups == g
constexpr int kConsumerWarps = kSliceWarps * kGroups;
// A stage must always be consumed by the same warps: a warp that waited on a stage it had not seen
// the previous phase of could pass try_wait.parity one phase early (parity aliasing).
static_assert(kStages % kGroups == 0, "a stage must belong to exactly one consumer group");
static_assert(kTileRows == kSliceWarps * 16, "one m16 slice per warp");
constexpr int kConsumerThreads = kConsumerWarps * 32;
constexpr int kMmaThreads = kConsumerThreads + 32;
constexpr int kTileBytes = kTileRows * kRowBytes;            // 16 KB per K or V tile
constexpr int kQBytes = kMaxGroup * kRowBytes;               // 2 KB
constexpr int kScratchFloats = kMaxGroup * kOStride + 2 * kMaxGroup;  // o[8][132], m[8], l[8]
constexpr int kFragFloats = 36 * 32;                         // o[32] + m[2] + l[2] per lane, [reg][lane]
static_assert(kFragFloats >= kScratchFloats, "the two merge layouts share one buffer");

struct __align__(128) SmemLayout {
  uint8_t kv[kStages][2][kTileBytes];
  uint8_t q[2][kQBytes];
  float scratch[kSliceWarps][kFragFloats];  // group merge (fragment layout), then slice merge (o[8][132], m, l)
  unsigned long long full_k[kStages], full_v[kStages], empty[kStages], q_full[2], q_empty[2];
  int meta[kStages][2];  // row_begin, row_end of the tile in each stage
  int nt[kMaxSeqsPerLaunch];
  int pre[kMaxSeqsPerLaunch + 1];
  int flag;
};

// ---- PTX wrappers ---------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(unsigned long long* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned long long* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, uint32_t parity) {
  const uint32_t a = smem_u32(bar);
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(a), "r"(parity) : "memory");
}
// 1-D bulk copy global -> shared, completion counted in bytes on an mbarrier (TMA engine).
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, unsigned long long* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}
// Same, with an L2 cache policy.  K/V rows are read once per step and never again before ~575 MB
// of other rows have gone by: evict_first keeps them from flushing the small hot state (tables,
// q, the rows the next step appends) out of the 126 MB L2.
__device__ __forceinline__ unsigned long long l2_policy_evict_first() {
  unsigned long long pol;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
  return pol;
}
__device__ __forceinline__ void bulk_g2s_hint(void* dst, const void* src, uint32_t bytes, unsigned long long* bar,
                                              unsigned long long pol) {
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(
          smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)), "l"(pol)
      : "memory");
}
__device__ __forceinline__ void ldsm_x4(uint32_t (&r)[4], uint32_t addr) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(addr));
}
__device__ __forceinline__ void ldsm_x4_t(uint32_t (&r)[4], uint32_t addr) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(addr));
}
__device__ __forceinline__ void mma_bf16(float (&d)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
  asm volatile(
      "mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
      : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
      : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
__device__ __forceinline__ uint32_t movmatrix_t(uint32_t x) {
  uint32_t y;
  asm volatile("movmatrix.sync.aligned.m8n8.trans.b16 %0, %1;" : "=r"(y) : "r"(x));
  return y;
}
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
  uint32_t r;
  asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
  return r;
}
__device__ __forceinline__ float ex2(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ unsigned smid() {
  unsigned r;
  asm volatile("mov.u32 %0, %%smid;" : "=r"(r));
  return r;
}
__device__ __forceinline__ void consumer_bar() { asm volatile("bar.sync 1, %0;" ::"n"(kConsumerThreads) : "memory"); }

// ---- walking the flattened (layer, seq, head, tile) list ---------------------------------------------
struct Cursor {
  int layer, i, h, k;  // layer index inside the call, index into the sequence list, KV head, tile
};

__device__ __forceinline__ Cursor locate(const SmemLayout& s, int n_seqs, int n_kv, long long x) {
  const long long per_layer = (long long)n_kv * s.pre[n_seqs];
  Cursor c;
  c.layer = (int)(x / per_layer);
  long long rem = x - (long long)c.layer * per_layer;
  int i = 0;
  while (i + 1 < n_seqs && (long long)n_kv * s.pre[i + 1] <= rem) ++i;
  rem -= (long long)n_kv * s.pre[i];
  c.i = i;
  c.h = (int)(rem / s.nt[i]);
  c.k = (int)(rem - (long long)c.h * s.nt[i]);
  return c;
}

__device__ __forceinline__ void next_item(const SmemLayout& s, int n_seqs, int n_kv, Cursor& c) {
  c.k = 0;
  if (++c.h < n_kv) return;
  c.h = 0;
  do {
    if (++c.i >= n_seqs) {
      c.i = 0;
      ++c.layer;
    }
  } while (s.nt[c.i] == 0);
}

struct AttnParams {
  const uint16_t* q;
  uint16_t* out;
  float* lse;
  int seq_base, n_seqs_total, layer_begin, n_layers_call;
  float sm_scale;
};

__global__ void __launch_bounds__(kMmaThreads, 1)
attn_mma_kernel(const __grid_constant__ CacheView c, const __grid_constant__ SeqList list,
                const __grid_constant__ AttnParams prm) {
  extern __shared__ __align__(128) uint8_t smem_raw[];
  SmemLayout& s = *reinterpret_cast<SmemLayout*>(smem_raw);
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int n_seqs = list.n, n_kv = c.n_kv, G = c.group;
  unsigned long long* trace = c.timeline + (size_t)blockIdx.x * kTimelineWords;
  pdl_launch_dependents();

  // ---- setup: barriers, tile counts, zeroed padding rows of the Q buffers ------------------------
  if (tid == 0) {
    for (int i = 0; i < kStages; ++i) {
      mbar_init(&s.full_k[i], 1);
      mbar_init(&s.full_v[i], 1);
      mbar_init(&s.empty[i], kSliceWarps);
    }
    for (int i = 0; i < 2; ++i) {
      mbar_init(&s.q_full[i], 1);
      mbar_init(&s.q_empty[i], kConsumerWarps);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  for (int i = tid; i < 2 * kQBytes / 4; i += kMmaThreads) reinterpret_cast<uint32_t*>(&s.q[0][0])[i] = 0u;
  // Everything above touches only this CTA's shared memory; from here on the kernel reads what
  // the step prologue (append + evict) wrote and writes buffers the previous launch may still use.
  pdl_wait();
  if (tid == 0) {
    trace[0] = globaltimer_ns();
    trace[1] = 0ull;
    trace[2] = smid();
    trace[3] = 0ull;
  }
  for (int i = tid; i < n_seqs; i += kMmaThreads) s.nt[i] = c.seqs[list.ids[i]].n_tiles;
  __syncthreads();
  if (tid == 0) {
    int acc = 0;
    for (int i = 0; i < n_seqs; ++i) {
      s.pre[i] = acc;
      acc += s.nt[i];
    }
    s.pre[n_seqs] = acc;
  }
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");  // zeroed Q rows vs later bulk copies
  __syncthreads();

  const long long total = (long long)prm.n_layers_call * n_kv * s.pre[n_seqs];
  const long long geff = total < (long long)gridDim.x ? total : (long long)gridDim.x;
  const long long cta = blockIdx.x;
  if (cta >= geff) return;
  const long long lo = cta * total / geff, hi = (cta + 1) * total / geff;

  const uint8_t* kpool = reinterpret_cast<const uint8_t*>(c.k_pool);
  const uint8_t* vpool = reinterpret_cast<const uint8_t*>(c.v_pool);

  if (warp == kConsumerWarps) {
    // =================================== producer warp ===================================
    // Walks its tile range in batches of <= 32 tiles of one item (lane j issues tile j); the
    // descriptors of the NEXT batch are loaded before the current one is issued, so their
    // global-load latency hides behind the copies.
    const unsigned long long kv_policy = l2_policy_evict_first();
    Cursor cur = locate(s, n_seqs, n_kv, lo);
    long long remaining = hi - lo;  // tiles left, counted from the start of the current item's segment
    int seg = (int)min((long long)(s.nt[cur.i] - cur.k), remaining);
    int base = 0, cnt = min(32, seg);
    uint32_t n = 0;  // tile sequence number of this CTA
    int item_no = 0;
    TileDesc td;
    if (lane < cnt) td = c.tiles[(size_t)list.ids[cur.i] * c.max_blocks + cur.k + lane];
    while (remaining > 0) {
      // ---- next batch (prefetch its descriptors) ----
      Cursor ncur = cur;
      int nseg = seg, nbase = base + cnt, ncnt = 0;
      long long nrem = remaining;
      const bool item_done = nbase >= seg;
      if (item_done) {
        nrem = remaining - seg;
        nbase = 0;
        if (nrem > 0) {
          next_item(s, n_seqs, n_kv, ncur);
          nseg = (int)min((long long)s.nt[ncur.i], nrem);
        }
      }
      if (nrem > 0) ncnt = min(32, nseg - nbase);
      TileDesc ntd;
      if (lane < ncnt) ntd = c.tiles[(size_t)list.ids[ncur.i] * c.max_blocks + ncur.k + nbase + lane];

      // ---- current batch ----
      const int layer = prm.layer_begin + cur.layer;
      if (base == 0 && lane == 0) {  // first batch of an item: stage its G query rows
        const int qb = item_no & 1;
        mbar_wait(&s.q_empty[qb], ((item_no >> 1) & 1) ^ 1);
        const size_t row = ((size_t)cur.layer * prm.n_seqs_total + prm.seq_base + cur.i) * c.n_q + (size_t)cur.h * G;
        mbar_expect_tx(&s.q_full[qb], (uint32_t)(G * kRowBytes));
        bulk_g2s(&s.q[qb][0], prm.q + row * kHeadDim, (uint32_t)(G * kRowBytes), &s.q_full[qb]);
      }
      for (int j = 0; j < cnt; ++j) {
        if (lane == j) {
          const uint32_t nn = n + (uint32_t)j;
          const int st = (int)(nn % kStages);
          const uint32_t ph = (nn / kStages) & 1u;
          mbar_wait(&s.empty[st], ph ^ 1u);
          s.meta[st][0] = td.row_begin;
          s.meta[st][1] = td.row_end;
          const uint32_t bytes = (uint32_t)(td.row_end - td.row_begin) * kRowBytes;
          mbar_expect_tx(&s.full_k[st], bytes);
          mbar_expect_tx(&s.full_v[st], bytes);
#pragma unroll
          for (int kv = 0; kv < 2; ++kv) {
            const uint8_t* pool = kv ? vpool : kpool;
            unsigned long long* bar = kv ? &s.full_v[st] : &s.full_k[st];
#pragma unroll
            for (int pg = 0; pg < 4; ++pg) {
              if (pg < td.n_pages) {
                const int r0 = (pg == 0) ? td.row_begin : pg * c.p;
                const int r1 = (pg == td.n_pages - 1) ? td.row_end : (pg + 1) * c.p;
                const uint8_t* src = pool + row_offset(c, layer, td.page[pg], cur.h, r0 - pg * c.p);
                bulk_g2s_hint(&s.kv[st][kv][r0 * kRowBytes], src, (uint32_t)(r1 - r0) * kRowBytes, bar, kv_policy);
              }
            }
          }
        }
        __syncwarp();
      }
      n += (uint32_t)cnt;
      if (item_done) {
        ++item_no;
        remaining = nrem;
      }
      cur = ncur;
      seg = nseg;
      base = nbase;
      cnt = ncnt;
      td = ntd;
    }
    return;
  }

  // ===================================== consumer warps =====================================
  // Warp (grp, w4): group grp takes every kGroups-th tile; inside a tile the warp owns rows
  // [16 w4, 16 w4 + 16).  All four warps of a group finish a tile within a few hundred cycles,
  // so a stage is handed back to the producer almost as soon as its data has landed and nearly
  // the whole ring stays in flight.  Each warp keeps its own online-softmax state (m, l, O^T)
  // over the rows it has seen; the states are merged at the end of the item.
  const float c2 = prm.sm_scale * 1.4426950408889634f;  // scores are kept raw; exp2((s - m) * c2)
  const int w4 = warp & (kSliceWarps - 1), grp = warp / kSliceWarps;
  const int lrow = lane >> 2;         // row inside an 8-row group / head index of B fragments
  const int lcol = (lane & 3) * 2;    // first of the two heads (or tokens) this lane owns
  // ldmatrix lane addressing (row inside the 16-row group, 16-byte chunk select, swizzle key)
  const int lm_row = ((lane >> 3) & 1) * 8 + (lane & 7);  // K (non-transposed): matrices 0..3 =
  const int lm_chk = lane >> 4;                           //   (rows 0-7, c), (8-15, c), (0-7, c+1), (8-15, c+1)
  const int lv_row = (lane >> 4) * 8 + (lane & 7);        // V (transposed): (rows 0-7, c), (0-7, c+1),
  const int lv_chk = (lane >> 3) & 1;                     //   (8-15, c), (8-15, c+1)
  const int key = lane & 7;
  const int slice0 = w4 * 16;                             // first row of this warp's slice
  const uint32_t k_off = (uint32_t)(slice0 + lm_row) * kRowBytes;
  const uint32_t v_off = (uint32_t)(slice0 + lv_row) * kRowBytes;

  Cursor cur = locate(s, n_seqs, n_kv, lo);
  long long remaining = hi - lo;
  long long pos = lo;
  uint32_t n = 0;
  int item_no = 0;
  bool first_segment = true;

  while (remaining > 0) {
    const int nt_i = s.nt[cur.i];
    const int seg = (int)min((long long)(nt_i - cur.k), remaining);
    const bool complete = (cur.k == 0) && (seg == nt_i);

    // ---- this item's query fragments (B operand of S^T = K Q^T) ----
    const int qb = item_no & 1;
    mbar_wait(&s.q_full[qb], (item_no >> 1) & 1);
    uint32_t qf[8][2];
    {
      const uint8_t* qs = &s.q[qb][0] + lrow * kRowBytes + lcol * 2;
#pragma unroll
      for (int ks = 0; ks < 8; ++ks) {
        qf[ks][0] = *reinterpret_cast<const uint32_t*>(qs + ks * 32);
        qf[ks][1] = *reinterpret_cast<const uint32_t*>(qs + ks * 32 + 16);
      }
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(&s.q_empty[qb]);

    float m0 = -INFINITY, m1 = -INFINITY, l0 = 0.f, l1 = 0.f;
    float o[8][4];
#pragma unroll
    for (int dt = 0; dt < 8; ++dt) o[dt][0] = o[dt][1] = o[dt][2] = o[dt][3] = 0.f;

    for (int tt = (grp + kGroups - (int)(n % kGroups)) % kGroups; tt < seg; tt += kGroups) {
      const uint32_t nn = n + (uint32_t)tt;
      const int st = (int)(nn % kStages);
      const uint32_t ph = (nn / kStages) & 1u;
      mbar_wait(&s.full_k[st], ph);
      const int rb = s.meta[st][0], re = s.meta[st][1];
      const bool act = (slice0 < re) && (slice0 + 16 > rb);  // warp-uniform: the slice holds valid rows
      uint32_t pb0 = 0u, pb1 = 0u;
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
        if (r0 < rb || r0 >= re) s0 = s1 = -INFINITY;
        if (r1 < rb || r1 >= re) s2 = s3 = -INFINITY;
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
        const bool edge = (slice0 < rb) || (slice0 + 16 > re);
        uint32_t mk01 = 0xffffffffu, mk23 = 0xffffffffu;
        if (edge) {  // rows outside [rb, re) were never copied: zero them in the A fragment
          const int t0 = slice0 + lcol;
          mk01 = ((t0 >= rb && t0 < re) ? 0x0000ffffu : 0u) | ((t0 + 1 >= rb && t0 + 1 < re) ? 0xffff0000u : 0u);
          mk23 = ((t0 + 8 >= rb && t0 + 8 < re) ? 0x0000ffffu : 0u) | ((t0 + 9 >= rb && t0 + 9 < re) ? 0xffff0000u : 0u);
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
    n += (uint32_t)seg;

    // ---- merge 1: groups 1.. hand their state to group 0 (same fragment layout, lane for lane) ----
#pragma unroll
    for (int r = 1; r < kGroups; ++r) {
      float* fs = s.scratch[w4];
      if (grp == r) {
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
      consumer_bar();
      if (grp == 0) {
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
      consumer_bar();
    }

    // ---- merge 2: the four row slices of group 0, through shared memory in [head][d] layout ----
    if (grp == 0) {
#pragma unroll
      for (int sh = 4; sh <= 16; sh <<= 1) {
        l0 += __shfl_xor_sync(0xffffffffu, l0, sh);
        l1 += __shfl_xor_sync(0xffffffffu, l1, sh);
      }
      float* my_scratch = s.scratch[w4];
#pragma unroll
      for (int dt = 0; dt < 8; ++dt) {
        const int d = dt * 16 + lrow;
        my_scratch[lcol * kOStride + d] = o[dt][0];
        my_scratch[(lcol + 1) * kOStride + d] = o[dt][1];
        my_scratch[lcol * kOStride + d + 8] = o[dt][2];
        my_scratch[(lcol + 1) * kOStride + d + 8] = o[dt][3];
      }
      if (lrow == 0) {
        my_scratch[kMaxGroup * kOStride + lcol] = m0;
        my_scratch[kMaxGroup * kOStride + lcol + 1] = m1;
        my_scratch[kMaxGroup * kOStride + kMaxGroup + lcol] = l0;
        my_scratch[kMaxGroup * kOStride + kMaxGroup + lcol + 1] = l1;
      }
    }
    consumer_bar();

    const int layer_c = cur.layer;
    const size_t out_row0 = ((size_t)layer_c * prm.n_seqs_total + prm.seq_base + cur.i) * c.n_q + (size_t)cur.h * G;
    // thread `tid` < 128 owns column d = tid of every head; the other consumer threads only sync
    const bool owner = tid < kHeadDim;
    const int col = owner ? tid : 0;
    float accv[kMaxGroup], Mh[kMaxGroup], Lh[kMaxGroup];
    if (owner) {
#pragma unroll
      for (int h = 0; h < kMaxGroup; ++h) {
        float M = -INFINITY;
#pragma unroll
        for (int w = 0; w < kSliceWarps; ++w) M = fmaxf(M, s.scratch[w][kMaxGroup * kOStride + h]);
        float L = 0.f, acc = 0.f;
#pragma unroll
        for (int w = 0; w < kSliceWarps; ++w) {
          const float mw = s.scratch[w][kMaxGroup * kOStride + h];
          const float f = (mw == -INFINITY) ? 0.f : ex2((mw - M) * c2);
          L += s.scratch[w][kMaxGroup * kOStride + kMaxGroup + h] * f;
          acc += s.scratch[w][h * kOStride + col] * f;
        }
        accv[h] = acc; Mh[h] = M; Lh[h] = L;
      }
    }

    if (complete) {
#pragma unroll
      for (int h = 0; h < kMaxGroup; ++h) {
        if (h < G && owner) {
          prm.out[(out_row0 + h) * kHeadDim + tid] = __bfloat16_as_ushort(__float2bfloat16_rn(accv[h] / Lh[h]));
          if (prm.lse != nullptr && tid == 0) prm.lse[out_row0 + h] = Mh[h] * prm.sm_scale + __logf(Lh[h]);
        }
      }
    } else {
      // split item: publish this CTA's partial; the last contributor merges all of them.
      const long long item_lo = pos - cur.k;
      const long long c_first = ((item_lo + 1) * geff - 1) / total;
      const long long c_last = ((item_lo + nt_i) * geff - 1) / total;
      const int slot = 2 * (int)cta + (first_segment ? 0 : 1);
      float* part = c.partials + (size_t)slot * kPartialFloats;
      if (owner) {
#pragma unroll
        for (int h = 0; h < kMaxGroup; ++h) part[h * kOStride + tid] = accv[h];
      }
      if (tid == 0) {
#pragma unroll
        for (int h = 0; h < kMaxGroup; ++h) {
          part[kMaxGroup * kOStride + h] = Mh[h];
          part[kMaxGroup * kOStride + kMaxGroup + h] = Lh[h];
        }
      }
      __threadfence();
      consumer_bar();
      int* counter = c.item_counters + ((size_t)layer_c * n_seqs + cur.i) * n_kv + cur.h;
      if (tid == 0) {
        __threadfence();  // release: every thread's partial (ordered by the barrier) before the ticket
        const int old = atomicAdd(counter, 1);
        s.flag = (old == (int)(c_last - c_first));
      }
      consumer_bar();
      if (s.flag && owner) {
        __threadfence();
        float M[kMaxGroup], L[kMaxGroup], acc[kMaxGroup];
#pragma unroll
        for (int h = 0; h < kMaxGroup; ++h) { M[h] = -INFINITY; L[h] = 0.f; acc[h] = 0.f; }
        for (long long cc = c_first; cc <= c_last; ++cc) {
          const long long lo_cc = cc * total / geff;
          const int sl = 2 * (int)cc + ((cc == c_first && lo_cc < item_lo) ? 1 : 0);
          const float* pp = c.partials + (size_t)sl * kPartialFloats;
#pragma unroll
          for (int h = 0; h < kMaxGroup; ++h) {
            const float mw = __ldcg(pp + kMaxGroup * kOStride + h);
            const float lw = __ldcg(pp + kMaxGroup * kOStride + kMaxGroup + h);
            const float ow = __ldcg(pp + h * kOStride + tid);
            const float Mn = fmaxf(M[h], mw);
            const float fa = (M[h] == -INFINITY) ? 0.f : ex2((M[h] - Mn) * c2);
            const float fb = (mw == -INFINITY) ? 0.f : ex2((mw - Mn) * c2);
            L[h] = L[h] * fa + lw * fb;
            acc[h] = acc[h] * fa + ow * fb;
            M[h] = Mn;
          }
        }
#pragma unroll
        for (int h = 0; h < kMaxGroup; ++h) {
          if (h < G) {
            prm.out[(out_row0 + h) * kHeadDim + tid] = __bfloat16_as_ushort(__float2bfloat16_rn(acc[h] / L[h]));
            if (prm.lse != nullptr && tid == 0) prm.lse[out_row0 + h] = M[h] * prm.sm_scale + __logf(L[h]);
          }
        }
        if (tid == 0) *counter = 0;  // self-resetting for the next launch
      }
    }
    consumer_bar();  // scratch and flag are reused by the next segment

    remaining -= seg;
    pos += seg;
    first_segment = false;
    ++item_no;
    next_item(s, n_seqs, n_kv, cur);
  }
  if (tid == 0) {
    trace[1] = globaltimer_ns();
    trace[3] = (unsigned long long)(hi - lo);
  }
}

}  // namespace

cudaError_t launch_attn_mma(const CacheView& c, const SeqList& list, int seq_base, int n_seqs_total, const void* q,
                            void* out, float* lse, int layer_begin, int layer_end, float sm_scale, int grid,
                            bool pdl, cudaStream_t st, LaunchInfo* info) {
  static bool attr_set = false;
  const int smem = (int)sizeof(SmemLayout);
  if (!attr_set) {
    cudaError_t e = cudaFuncSetAttribute(attn_mma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e != cudaSuccess) return e;
    attr_set = true;
  }
  if (grid > kMaxAttnGrid) grid = kMaxAttnGrid;
  AttnParams prm;
  prm.q = reinterpret_cast<const uint16_t*>(q);
  prm.out = reinterpret_cast<uint16_t*>(out);
  prm.lse = lse;
  prm.seq_base = seq_base;
  prm.n_seqs_total = n_seqs_total;
  prm.layer_begin = layer_begin;
  prm.n_layers_call = layer_end - layer_begin;
  prm.sm_scale = sm_scale;
  PdlLaunch l(dim3((unsigned)grid), dim3(kMmaThreads), (size_t)smem, st, pdl);
  info->launches += 1;
  info->grid = grid;
  info->smem = smem;
  return cudaLaunchKernelEx(&l.cfg, attn_mma_kernel, c, list, prm);
}

}  // namespace murmur
