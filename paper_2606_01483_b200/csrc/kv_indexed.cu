// General index-set eviction with dense stable compaction ("indexed mode").
//
// "the evictable tokens are not contiguous and cannot be captured by a simple positional
// policy. This motivates future work on adaptive speech token selection strategies, such as query-aware ...
// eviction policies"; the sparsity it measures is per layer and head.  This file is
// that future work's cache side: per-(layer, KV head) retained index sets, applied by a dense, stable,
// IN-PLACE compaction (slot s of a slab <- row of the s-th smallest retained position), a head-ragged
// append, and Eq. 1 over the slabs.  Definitions: DESIGN.md "f3" (a convention of this
// build - the paper defines none).
//
// In-place compaction of one slab (layer, head): rows only move towards lower linear addresses (the s-th
// smallest retained position has at least s resident rows below it), so chunks of 64 destination slots are
// processed in ascending order - all source rows of a chunk are loaded into registers, one barrier, then
// stored; later chunks read strictly behind earlier chunks' writes.  One CTA per slab; slabs never share
// bytes (a page holds every layer's and head's rows of a block, each in its own 256-byte-row region).
// Rows are re-swizzled on the way (the pool keeps chunk c of slot s at c ^ (s & 7)).
#include <cuda_bf16.h>

#include "device_state.cuh"

namespace murmur {
namespace {

constexpr int kIdxThreads = 256;
constexpr int kIdxChunk = 64;  // destination slots per pass: 16 half-warps x 4 rows

__device__ __forceinline__ void idx_error(const CacheView& c, int code) { atomicCAS(&c.ctrl[kCtrlError], 0, code); }

// largest index i in [0, n) with a[i] <= x (a ascending), or -1
__device__ __forceinline__ int upper_index(const int32_t* a, int n, int x) {
  int lo = -1, hi = n - 1;
  while (lo < hi) {
    const int mid = (lo + hi + 1) >> 1;
    if (a[mid] <= x) lo = mid; else hi = mid - 1;
  }
  return lo;
}

__global__ void __launch_bounds__(kIdxThreads)
indexed_defrag_kernel(const __grid_constant__ CacheView c, const __grid_constant__ IdxView ix, int seq,
                      const int32_t* __restrict__ sel_pos, const int32_t* __restrict__ sel_cnt, int cap_sel,
                      int from_positional, unsigned long long* __restrict__ moved) {
  const int slab = blockIdx.x;  // layer * n_kv + head
  const int layer = slab / c.n_kv, head = slab % c.n_kv;
  const int tid = threadIdx.x, sub = tid & 15, hw = tid >> 4;
  const int p = c.p, plog = c.p_log2;
  const SeqDev& sd = c.seqs[seq];
  const int32_t* sel = sel_pos + (size_t)slab * cap_sel;
  const int n_new = sel_cnt[slab];
  int32_t* len_p = ix.len + (size_t)seq * c.n_layers * c.n_kv + slab;
  int32_t* pos = ix.pos + ((size_t)seq * c.n_layers * c.n_kv + slab) * ix.cap;
  const int n_old = from_positional ? 0 : *len_p;
  const int32_t* tab = c.block_table + (size_t)seq * c.max_blocks;
  const int32_t* lpages = c.live_pages + (size_t)seq * c.max_blocks;
  const int32_t* lblocks = c.live_blocks + (size_t)seq * c.max_blocks;
  const int n_live = sd.n_live;
  if (n_new < 1 || n_new > cap_sel || n_new > ix.cap) {
    if (tid == 0) idx_error(c, 1);
    return;
  }
  uint8_t* kp = reinterpret_cast<uint8_t*>(c.k_pool);
  uint8_t* vp = reinterpret_cast<uint8_t*>(c.v_pool);
  unsigned long long n_moved = 0;
  for (int s0 = 0; s0 < n_new; s0 += kIdxChunk) {
    uint4 kv[4][2];
    int dst_page[4], ok[4];
#pragma unroll
    for (int r = 0; r < 4; ++r) {
      const int s = s0 + hw + 16 * r;
      ok[r] = 0;
      dst_page[r] = -1;
      if (s < n_new) {
        const int x = sel[s];
        int src_page = -1, src_slot = 0;
        if (s > 0 && sel[s - 1] >= x) idx_error(c, 1);  // not strictly ascending
        if (from_positional) {  // position x lives in logical block x >> plog, which must be live
          const int k = upper_index(lblocks, n_live, x >> plog);
          if (x >= 0 && x < sd.len && k >= 0 && lblocks[k] == (x >> plog)) {
            src_page = lpages[k];
            src_slot = x & (p - 1);
          }
          dst_page[r] = (s >> plog) < n_live ? lpages[s >> plog] : -1;
        } else {  // position x is the row in the slot where pos[] holds x
          const int so = upper_index(pos, n_old, x);
          if (so >= 0 && pos[so] == x) {
            src_page = tab[so >> plog];
            src_slot = so & (p - 1);
          }
          dst_page[r] = (s >> plog) < sd.idx_blocks ? tab[s >> plog] : -1;
        }
        if (src_page < 0 || dst_page[r] < 0) {
          if (sub == 0) idx_error(c, 2);  // a selected position is not held by this slab
        } else {
          ok[r] = 1;
          const size_t off = row_offset(c, layer, src_page, head, src_slot) + (size_t)((sub ^ (src_slot & 7)) << 4);
          kv[r][0] = *reinterpret_cast<const uint4*>(kp + off);
          kv[r][1] = *reinterpret_cast<const uint4*>(vp + off);
          if (sub == 0 && (src_page != dst_page[r] || src_slot != (s & (p - 1)))) ++n_moved;
        }
      }
    }
    __syncthreads();  // every source row of this chunk is in registers
#pragma unroll
    for (int r = 0; r < 4; ++r) {
      const int s = s0 + hw + 16 * r;
      if (ok[r]) {
        const int slot = s & (p - 1);
        const size_t off = row_offset(c, layer, dst_page[r], head, slot) + (size_t)((sub ^ (slot & 7)) << 4);
        *reinterpret_cast<uint4*>(kp + off) = kv[r][0];
        *reinterpret_cast<uint4*>(vp + off) = kv[r][1];
      }
    }
  }
  __syncthreads();  // all look-ups through the old position table are done
  for (int s = tid; s < n_new; s += kIdxThreads) pos[s] = sel[s];
  if (tid == 0) *len_p = n_new;
  if (sub == 0 && n_moved) atomicAdd(moved, n_moved);
}

// Read-only check of the index sets before anything moves: every set has 1 .. min(cap_sel, table capacity) elements,
// is strictly ascending, names only positions its slab holds, and fits the blocks the sequence keeps.  The first
// violation's code lands in *bad (1 = size / order, 2 = a position that is not held); the defrag is launched only when
// the host has read 0 there - an in-place compaction cannot be undone once rows have been overwritten.
__global__ void __launch_bounds__(kIdxThreads)
indexed_validate_kernel(const __grid_constant__ CacheView c, const __grid_constant__ IdxView ix, int seq,
                        const int32_t* __restrict__ sel_pos, const int32_t* __restrict__ sel_cnt, int cap_sel,
                        int from_positional, int* __restrict__ bad) {
  const int slab = blockIdx.x;
  const int plog = c.p_log2;
  const SeqDev& sd = c.seqs[seq];
  const int32_t* sel = sel_pos + (size_t)slab * cap_sel;
  const int n_new = sel_cnt[slab];
  if (n_new < 1 || n_new > cap_sel || n_new > ix.cap) {
    if (threadIdx.x == 0) atomicCAS(bad, 0, 1);
    return;
  }
  const int32_t* pos = ix.pos + ((size_t)seq * c.n_layers * c.n_kv + slab) * ix.cap;
  const int n_old = from_positional ? 0 : ix.len[(size_t)seq * c.n_layers * c.n_kv + slab];
  const int32_t* lblocks = c.live_blocks + (size_t)seq * c.max_blocks;
  const int n_live = sd.n_live;
  const int blocks_kept = from_positional ? n_live : sd.idx_blocks;
  if (((n_new - 1) >> plog) >= blocks_kept) {  // the last destination slot has no page
    if (threadIdx.x == 0) atomicCAS(bad, 0, 2);
    return;
  }
  int err = 0;
  for (int s = threadIdx.x; s < n_new; s += kIdxThreads) {
    const int x = sel[s];
    if (s > 0 && sel[s - 1] >= x) err = err ? err : 1;
    bool held;
    if (from_positional) {
      const int k = upper_index(lblocks, n_live, x >> plog);
      held = x >= 0 && x < sd.len && k >= 0 && lblocks[k] == (x >> plog);
    } else {
      const int so = upper_index(pos, n_old, x);
      held = so >= 0 && pos[so] == x;
    }
    if (!held) err = err ? err : 2;
  }
  if (err) atomicCAS(bad, 0, err);
}

// After the slabs: keep blocks 0 .. ceil(max len / p) - 1, push the surplus pages (ascending), switch the mode.
__global__ void indexed_commit_kernel(const __grid_constant__ CacheView c, const __grid_constant__ IdxView ix, int seq,
                                      int from_positional) {
  __shared__ int s_max;
  SeqDev& sd = c.seqs[seq];
  const int n_slabs = c.n_layers * c.n_kv;
  const int32_t* len = ix.len + (size_t)seq * n_slabs;
  if (threadIdx.x == 0) s_max = 0;
  __syncthreads();
  int mx = 0;
  for (int i = threadIdx.x; i < n_slabs; i += blockDim.x) mx = max(mx, len[i]);
  atomicMax(&s_max, mx);
  __syncthreads();
  if (threadIdx.x != 0) return;
  const int nb_new = (s_max + c.p - 1) >> c.p_log2;
  int32_t* tab = c.block_table + (size_t)seq * c.max_blocks;
  int top = c.ctrl[kCtrlFreeTop];
  if (from_positional) {
    const int32_t* lpages = c.live_pages + (size_t)seq * c.max_blocks;
    const int n_live = sd.n_live;
    const int n_tab = (sd.len + c.p - 1) >> c.p_log2;
    for (int k = nb_new; k < n_live; ++k) c.free_stack[top++] = lpages[k];
    for (int k = 0; k < n_tab || k < nb_new; ++k) tab[k] = k < nb_new ? lpages[k] : -1;
    sd.idx_next_pos = sd.len;
    sd.idx_mode = 1;
    sd.n_runs = 0; sd.n_tiles = 0; sd.n_retained = 0; sd.n_live = nb_new;
    sd.tg_len[0] = sd.tg_len[1] = -1;
  } else {
    for (int k = nb_new; k < sd.idx_blocks; ++k) {
      c.free_stack[top++] = tab[k];
      tab[k] = -1;
    }
  }
  c.ctrl[kCtrlFreeTop] = top;
  sd.idx_blocks = nb_new;
  sd.idx_max_len = s_max;
}

// ---- append: one token per listed sequence, to every slab ------------------------------------------------
__global__ void indexed_alloc_kernel(const __grid_constant__ CacheView c, const __grid_constant__ SeqList list) {
  if (threadIdx.x != 0) return;
  int top = c.ctrl[kCtrlFreeTop];
  for (int i = 0; i < list.n; ++i) {  // call order (allocator C3)
    SeqDev& sd = c.seqs[list.ids[i]];
    if (!sd.active || !sd.idx_mode) {
      idx_error(c, 2);
      continue;
    }
    if (((sd.idx_max_len + c.p) >> c.p_log2) > sd.idx_blocks) {  // the longest slab starts a new block
      if (top < 1 || sd.idx_blocks >= c.max_blocks) {
        idx_error(c, 3);
        continue;
      }
      c.block_table[(size_t)list.ids[i] * c.max_blocks + sd.idx_blocks] = c.free_stack[--top];
      sd.idx_blocks += 1;
    }
  }
  c.ctrl[kCtrlFreeTop] = top;
}

__global__ void __launch_bounds__(kIdxThreads)
indexed_scatter_kernel(const __grid_constant__ CacheView c, const __grid_constant__ IdxView ix,
                       const __grid_constant__ SeqList list, const uint4* __restrict__ k_new, const uint4* __restrict__ v_new) {
  const int sub = threadIdx.x & 15;
  const int n_slabs = c.n_layers * c.n_kv;
  const long long rows = (long long)n_slabs * list.n;  // per K / per V: [layer][seq][head]
  const long long stride = (long long)gridDim.x * (kIdxThreads / 16);
  for (long long u = (long long)blockIdx.x * (kIdxThreads / 16) + (threadIdx.x >> 4); u < 2 * rows; u += stride) {
    const int is_v = u >= rows;
    const long long r = is_v ? u - rows : u;
    const int head = (int)(r % c.n_kv);
    const int i = (int)((r / c.n_kv) % list.n);
    const int layer = (int)(r / ((long long)c.n_kv * list.n));
    const int id = list.ids[i];
    const int slab = layer * c.n_kv + head;
    const int slot_lin = ix.len[(size_t)id * n_slabs + slab];  // bumped by the next kernel
    const int page = (slot_lin >> c.p_log2) < c.max_blocks ? c.block_table[(size_t)id * c.max_blocks + (slot_lin >> c.p_log2)] : -1;
    if (page < 0 || slot_lin >= ix.cap) {
      if (sub == 0) idx_error(c, 2);
      continue;
    }
    const int slot = slot_lin & (c.p - 1);
    uint8_t* pool = reinterpret_cast<uint8_t*>(is_v ? c.v_pool : c.k_pool);
    *reinterpret_cast<uint4*>(pool + row_offset(c, layer, page, head, slot) + (size_t)((sub ^ (slot & 7)) << 4)) =
        (is_v ? v_new : k_new)[r * 16 + sub];
  }
}

__global__ void indexed_bump_kernel(const __grid_constant__ CacheView c, const __grid_constant__ IdxView ix,
                                    const __grid_constant__ SeqList list) {
  const int n_slabs = c.n_layers * c.n_kv;
  const int i = blockIdx.x;
  const int id = list.ids[i];
  SeqDev& sd = c.seqs[id];
  for (int slab = threadIdx.x; slab < n_slabs; slab += blockDim.x) {
    int32_t* len = ix.len + (size_t)id * n_slabs + slab;
    const int s = *len;
    if (s < ix.cap) {
      ix.pos[((size_t)id * n_slabs + slab) * ix.cap + s] = sd.idx_next_pos;
      *len = s + 1;
    }
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    sd.idx_next_pos += 1;
    sd.idx_max_len += 1;
  }
}

__global__ void indexed_seq_end_kernel(const __grid_constant__ CacheView c, int seq) {
  if (threadIdx.x != 0) return;
  SeqDev& sd = c.seqs[seq];
  int32_t* tab = c.block_table + (size_t)seq * c.max_blocks;
  int top = c.ctrl[kCtrlFreeTop];
  for (int k = 0; k < sd.idx_blocks; ++k) {
    c.free_stack[top++] = tab[k];
    tab[k] = -1;
  }
  c.ctrl[kCtrlFreeTop] = top;
  sd.active = 0; sd.len = 0; sd.idx_mode = 0; sd.idx_blocks = 0; sd.idx_max_len = 0; sd.n_live = 0;
}

// ---- attention over the slabs: Eq. 1 of query head hq over the rows of slab (layer, hq / G) ----------------
// First path: FFMA straight from the pool (the structure of decode_attn_generic.cu; rows are dense, so
// row j of the slab is slot j of the sequence's blocks).  One CTA per (layer, sequence, KV head).
constexpr int kIaWarps = 8;

__device__ __forceinline__ float bf_lo16(uint32_t w) { return __uint_as_float(w << 16); }
__device__ __forceinline__ float bf_hi16(uint32_t w) { return __uint_as_float(w & 0xffff0000u); }

__global__ void __launch_bounds__(kIaWarps * 32)
indexed_attn_kernel(const __grid_constant__ CacheView c, const __grid_constant__ IdxView ix,
                    const __grid_constant__ SeqList list, const uint16_t* __restrict__ q, uint16_t* __restrict__ out,
                    float* __restrict__ lse, float sm_scale) {
  __shared__ float s_m[kIaWarps][kMaxGroup];
  __shared__ float s_l[kIaWarps][kMaxGroup];
  __shared__ float s_o[kIaWarps][kMaxGroup][kHeadDim];
  const int g = blockIdx.x, i = blockIdx.y, layer = blockIdx.z;
  const int id = list.ids[i];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int G = c.group;
  const int n = ix.len[(size_t)id * c.n_layers * c.n_kv + layer * c.n_kv + g];
  const int32_t* tab = c.block_table + (size_t)id * c.max_blocks;
  const size_t q_row0 = ((size_t)layer * list.n + i) * c.n_q + (size_t)g * G;
  float qv[kMaxGroup][4];
#pragma unroll
  for (int h = 0; h < kMaxGroup; ++h) {
    if (h < G) {
      const uint2 w = reinterpret_cast<const uint2*>(q + (q_row0 + h) * kHeadDim)[lane];
      qv[h][0] = bf_lo16(w.x); qv[h][1] = bf_hi16(w.x); qv[h][2] = bf_lo16(w.y); qv[h][3] = bf_hi16(w.y);
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
  const int chunk = lane >> 1, half = lane & 1;
  for (int j = warp; j < n; j += kIaWarps) {
    const int page = tab[j >> c.p_log2];
    const int slot = j & (c.p - 1);
    const size_t off = row_offset(c, layer, page, g, slot) + (size_t)((chunk ^ (slot & 7)) * 16 + half * 8);
    const uint2 kw = *reinterpret_cast<const uint2*>(kp + off);
    const uint2 vw = *reinterpret_cast<const uint2*>(vp + off);
    const float k0 = bf_lo16(kw.x), k1 = bf_hi16(kw.x), k2 = bf_lo16(kw.y), k3 = bf_hi16(kw.y);
    const float v0 = bf_lo16(vw.x), v1 = bf_hi16(vw.x), v2 = bf_lo16(vw.y), v3 = bf_hi16(vw.y);
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
  for (int e = threadIdx.x; e < G * kHeadDim; e += kIaWarps * 32) {
    const int h = e / kHeadDim, d = e % kHeadDim;
    float M = -INFINITY;
#pragma unroll
    for (int w = 0; w < kIaWarps; ++w) M = fmaxf(M, s_m[w][h]);
    float L = 0.f, acc = 0.f;
#pragma unroll
    for (int w = 0; w < kIaWarps; ++w) {
      const float sc = (s_m[w][h] == -INFINITY) ? 0.f : __expf(s_m[w][h] - M);
      L += s_l[w][h] * sc;
      acc += s_o[w][h][d] * sc;
    }
    const size_t orow = q_row0 + h;
    out[orow * kHeadDim + d] = __bfloat16_as_ushort(__float2bfloat16_rn(acc / L));
    if (lse != nullptr && d == 0) lse[orow] = M + __logf(L);
  }
}

// ---- introspection: the rows of every slab, by slot, natural (un-swizzled) order ------------------------------
__global__ void indexed_gather_kernel(const __grid_constant__ CacheView c, const __grid_constant__ IdxView ix, int seq,
                                      uint4* __restrict__ k_out, uint4* __restrict__ v_out, int cap_out) {
  const int sub = threadIdx.x & 15;
  const int n_slabs = c.n_layers * c.n_kv;
  const long long rows = (long long)n_slabs * cap_out;
  const long long stride = (long long)gridDim.x * (blockDim.x / 16);
  for (long long r = (long long)blockIdx.x * (blockDim.x / 16) + (threadIdx.x >> 4); r < rows; r += stride) {
    const int s = (int)(r % cap_out), slab = (int)(r / cap_out);
    const int layer = slab / c.n_kv, head = slab % c.n_kv;
    uint4 kvv = make_uint4(0u, 0u, 0u, 0u), vvv = kvv;
    if (s < ix.len[(size_t)seq * n_slabs + slab]) {
      const int page = c.block_table[(size_t)seq * c.max_blocks + (s >> c.p_log2)];
      const int slot = s & (c.p - 1);
      if (page >= 0) {
        const size_t off = row_offset(c, layer, page, head, slot) + (size_t)((sub ^ (slot & 7)) << 4);
        kvv = *reinterpret_cast<const uint4*>(reinterpret_cast<const uint8_t*>(c.k_pool) + off);
        vvv = *reinterpret_cast<const uint4*>(reinterpret_cast<const uint8_t*>(c.v_pool) + off);
      } else if (sub == 0) {
        idx_error(c, 2);
      }
    }
    k_out[r * 16 + sub] = kvv;
    v_out[r * 16 + sub] = vvv;
  }
}

// ---- producer of query-aware sets: membership mask -> ascending position lists ------------------------------------
// One CTA per slab.  keep(x) = resident and (mask[x] or system prompt or among the n_recent newest).
__global__ void __launch_bounds__(kIdxThreads)
select_compact_kernel(const __grid_constant__ CacheView c, int seq, const uint8_t* __restrict__ mask, long long mask_stride,
                      int n_recent, int32_t* __restrict__ sel_pos, int32_t* __restrict__ sel_cnt, int cap_sel) {
  __shared__ int s_scan[kIdxThreads + 1];
  const int slab = blockIdx.x, tid = threadIdx.x;
  const SeqParams sp = load_params(c.seqs[seq]);
  const int len = sp.len;
  Interval dead[2];
  const int n_dead = dead_intervals(sp, dead);
  const int32_t* tab = c.block_table + (size_t)seq * c.max_blocks;
  const uint8_t* mk = mask + (size_t)slab * mask_stride;
  const int per = (len + kIdxThreads - 1) / kIdxThreads;
  const int x0 = min(len, tid * per), x1 = min(len, x0 + per);
  auto keep = [&](int x) {
    bool is_dead = false;
    for (int k = 0; k < n_dead; ++k) is_dead |= (x >= dead[k].a && x < dead[k].b);
    if (is_dead || tab[x >> c.p_log2] < 0) return false;
    return mk[x] != 0 || x < sp.P || (x >= sp.P + sp.S && x < sp.P + sp.S + sp.M) || x >= len - n_recent;
  };
  int cnt = 0;
  for (int x = x0; x < x1; ++x) cnt += keep(x) ? 1 : 0;
  s_scan[tid + 1] = cnt;
  if (tid == 0) s_scan[0] = 0;
  __syncthreads();
  if (tid == 0)
    for (int k = 1; k <= kIdxThreads; ++k) s_scan[k] += s_scan[k - 1];
  __syncthreads();
  int rank = s_scan[tid];
  int32_t* dst = sel_pos + (size_t)slab * cap_sel;
  for (int x = x0; x < x1; ++x)
    if (keep(x)) {
      if (rank < cap_sel) dst[rank] = x;
      ++rank;
    }
  if (tid == 0) {
    sel_cnt[slab] = s_scan[kIdxThreads];
    if (s_scan[kIdxThreads] > cap_sel) idx_error(c, 1);
  }
}

}  // namespace

cudaError_t launch_indexed_validate(const CacheView& c, const IdxView& ix, int seq, const int32_t* sel_pos,
                                    const int32_t* sel_cnt, int cap_sel, bool from_positional, int* bad_dev,
                                    cudaStream_t st, LaunchInfo* info) {
  indexed_validate_kernel<<<c.n_layers * c.n_kv, kIdxThreads, 0, st>>>(c, ix, seq, sel_pos, sel_cnt, cap_sel,
                                                                       from_positional ? 1 : 0, bad_dev);
  info->launches += 1;
  return cudaGetLastError();
}

cudaError_t launch_indexed_defrag(const CacheView& c, const IdxView& ix, int seq, const int32_t* sel_pos, const int32_t* sel_cnt,
                                  int cap_sel, bool from_positional, unsigned long long* moved_dev, cudaStream_t st,
                                  LaunchInfo* info) {
  indexed_defrag_kernel<<<c.n_layers * c.n_kv, kIdxThreads, 0, st>>>(c, ix, seq, sel_pos, sel_cnt, cap_sel,
                                                                     from_positional ? 1 : 0, moved_dev);
  indexed_commit_kernel<<<1, 128, 0, st>>>(c, ix, seq, from_positional ? 1 : 0);
  info->launches += 2;
  info->grid = c.n_layers * c.n_kv;
  return cudaGetLastError();
}

cudaError_t launch_indexed_append(const CacheView& c, const IdxView& ix, const SeqList& list, const void* k_new,
                                  const void* v_new, cudaStream_t st, LaunchInfo* info) {
  indexed_alloc_kernel<<<1, 32, 0, st>>>(c, list);
  const long long units = 2LL * c.n_layers * c.n_kv * list.n;
  long long grid = (units + 15) / 16;
  if (grid > 1024) grid = 1024;
  indexed_scatter_kernel<<<(int)grid, kIdxThreads, 0, st>>>(c, ix, list, reinterpret_cast<const uint4*>(k_new),
                                                            reinterpret_cast<const uint4*>(v_new));
  indexed_bump_kernel<<<list.n, 128, 0, st>>>(c, ix, list);
  info->launches += 3;
  info->grid = (int)grid;
  return cudaGetLastError();
}

cudaError_t launch_indexed_attn(const CacheView& c, const IdxView& ix, const SeqList& list, const void* q, void* out,
                                float* lse, float sm_scale, cudaStream_t st, LaunchInfo* info) {
  dim3 grid(c.n_kv, list.n, c.n_layers);
  indexed_attn_kernel<<<grid, kIaWarps * 32, 0, st>>>(c, ix, list, reinterpret_cast<const uint16_t*>(q),
                                                      reinterpret_cast<uint16_t*>(out), lse, sm_scale);
  info->launches += 1;
  info->grid = (int)(grid.x * grid.y * grid.z);
  return cudaGetLastError();
}

cudaError_t launch_indexed_gather(const CacheView& c, const IdxView& ix, int seq, void* k_out, void* v_out, int cap_out,
                                  cudaStream_t st, LaunchInfo* info) {
  const long long rows = (long long)c.n_layers * c.n_kv * cap_out;
  long long grid = (rows + 15) / 16;
  if (grid > 4096) grid = 4096;
  if (grid < 1) grid = 1;
  indexed_gather_kernel<<<(int)grid, 256, 0, st>>>(c, ix, seq, reinterpret_cast<uint4*>(k_out), reinterpret_cast<uint4*>(v_out),
                                                   cap_out);
  info->launches += 1;
  return cudaGetLastError();
}

cudaError_t launch_indexed_seq_end(const CacheView& c, int seq, cudaStream_t st, LaunchInfo* info) {
  indexed_seq_end_kernel<<<1, 32, 0, st>>>(c, seq);
  info->launches += 1;
  return cudaGetLastError();
}

cudaError_t launch_select_compact(const CacheView& c, int seq, const uint8_t* mask, long long mask_stride, int n_recent,
                                  int32_t* sel_pos, int32_t* sel_cnt, int cap_sel, cudaStream_t st, LaunchInfo* info) {
  select_compact_kernel<<<c.n_layers * c.n_kv, kIdxThreads, 0, st>>>(c, seq, mask, mask_stride, n_recent, sel_pos, sel_cnt,
                                                                     cap_sel);
  info->launches += 1;
  return cudaGetLastError();
}

}  // namespace murmur
