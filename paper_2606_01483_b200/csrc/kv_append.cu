// murmur_kv_append and the small state kernels (init, seq_begin, seq_end, gather, expand).
//
// append (the cache C receives the K,V of decode step j; prefill uses the
// same call): ONE kernel.  Every CTA recomputes the (tiny) page allocation of the call from
// the old device state - an exclusive prefix sum of per-sequence new-block counts, pages popped
// from the top of the free stack in call order (C3) - scatters its share of the rows
// into the pre-swizzled pools, and the LAST CTA to finish (ticket counter) commits the new
// lengths, block-table entries and free-stack height.  No host sync, graph-capturable.
// With fuse_evict (the decode-step prologue) the eviction for the same sequences rides along:
// its table products are computed by warps of all CTAs before the ticket, and the last CTA only
// frees the dead pages after the commit - append -> evict is one launch.
#include "evict_body.cuh"

namespace murmur {
namespace {

__device__ __forceinline__ void set_error(const CacheView& c, int code) { atomicCAS(&c.ctrl[kCtrlError], 0, code); }

__global__ void init_kernel(CacheView c, int n_counters) {
  const size_t tid = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (size_t i = tid; i < (size_t)c.n_pages; i += stride) c.free_stack[i] = (int32_t)(c.n_pages - 1 - i);
  const size_t n_tab = (size_t)c.max_seqs * c.max_blocks;
  for (size_t i = tid; i < n_tab; i += stride) {
    c.block_table[i] = -1;
    c.live_pages[i] = -1;
    c.live_blocks[i] = -1;
  }
  int32_t* seq_words = reinterpret_cast<int32_t*>(c.seqs);
  for (size_t i = tid; i < (size_t)c.max_seqs * (sizeof(SeqDev) / 4); i += stride) seq_words[i] = 0;
  for (size_t i = tid; i < (size_t)n_counters; i += stride) c.item_counters[i] = 0;
  if (tid < kCtrlWords) c.ctrl[tid] = (tid == kCtrlFreeTop) ? (int32_t)c.n_pages : 0;
}

__global__ void seq_begin_kernel(CacheView c, int seq, SeqParams sp) {
  int32_t* tab = c.block_table + (size_t)seq * c.max_blocks;
  for (int b = threadIdx.x; b < c.max_blocks; b += blockDim.x) tab[b] = -1;
  if (threadIdx.x == 0) {
    SeqDev& s = c.seqs[seq];
    if (s.active) set_error(c, 2);
    s.P = sp.P; s.S = sp.S; s.M = sp.M; s.len = 0;
    s.w_s = sp.w_s; s.d = sp.d; s.k_s = sp.k_s; s.w_o = sp.w_o; s.k_o = sp.k_o;
    s.active = 1;
    s.n_live = 0; s.n_runs = 0; s.n_tiles = 0; s.n_retained = 0;
    s.tg_len[0] = s.tg_len[1] = -1;
    s.idx_mode = 0; s.idx_blocks = 0; s.idx_next_pos = 0; s.idx_max_len = 0;
  }
}

// One warp: pushes the live blocks of `seq` in ascending logical order, then deactivates it.
__global__ void seq_end_kernel(CacheView c, int seq) {
  const int lane = threadIdx.x;
  SeqDev& s = c.seqs[seq];
  if (!s.active) {
    if (lane == 0) set_error(c, 2);
    return;
  }
  int32_t* tab = c.block_table + (size_t)seq * c.max_blocks;
  const int nblk = (s.len + c.p - 1) >> c.p_log2;
  const int top = c.ctrl[kCtrlFreeTop];
  int run = 0;
  for (int b0 = 0; b0 < nblk; b0 += 32) {
    const int b = b0 + lane;
    const int pg = (b < nblk) ? tab[b] : -1;
    const unsigned m = __ballot_sync(0xffffffffu, pg >= 0);
    if (pg >= 0) {
      c.free_stack[top + run + __popc(m & ((1u << lane) - 1))] = pg;
      tab[b] = -1;
    }
    run += __popc(m);
  }
  __syncwarp();
  if (lane == 0) {
    c.ctrl[kCtrlFreeTop] = top + run;
    s.active = 0;
    s.len = 0;
    s.n_live = 0; s.n_runs = 0; s.n_tiles = 0; s.n_retained = 0;
  }
}

// ---- append -----------------------------------------------------------------------------------
constexpr int kAppendThreads = 256;  // small enough to be co-resident with an attention CTA (registers)

// One half-warp moves one 256-byte row (16 lanes x 16 bytes).  Unit u of a call = (K|V, layer, token, head).
struct RowUnit {
  const uint4* src;
  int page;               // loaded, not yet consumed: dst() is the first use
  int is_v;
  size_t off0;            // byte offset of the destination chunk in a pool, without the page term
  __device__ __forceinline__ uint4* dst(const CacheView& c) const {
    uint8_t* pool = reinterpret_cast<uint8_t*>(is_v ? c.v_pool : c.k_pool);
    return reinterpret_cast<uint4*>(pool + off0 + (size_t)page * ((size_t)c.n_kv * c.p * kRowBytes));
  }
};

// page: >= 0 the row's physical page; kRowBad = a position that should be mapped is not (device error);
// kRowSkip = nothing to store (no row, or - write-only calls - a position the eviction has already freed).
constexpr int kRowBad = -1, kRowSkip = -2;

__device__ __forceinline__ RowUnit locate_row(const CacheView& c, const AppendList& list, long long u, long long rows_src,
                                              int total_tokens, int layer_begin, int n, int free_top, int sub,
                                              const uint4* k_new, const uint4* v_new, const int* s_tok_off,
                                              const int* s_blk_off, const int* s_old_nblk, const SeqParams* s_sp,
                                              bool reserve) {
  const int is_v = u >= rows_src;
  const long long r = is_v ? u - rows_src : u;
  int head, tau, layer;
  if (rows_src < 0x7fffffffLL) {  // 32-bit index arithmetic (64-bit division is ~100 instructions)
    const unsigned r32 = (unsigned)r, r2 = r32 / (unsigned)c.n_kv;
    head = (int)(r32 - r2 * (unsigned)c.n_kv);
    const unsigned lq = r2 / (unsigned)total_tokens;
    tau = (int)(r2 - lq * (unsigned)total_tokens);
    layer = layer_begin + (int)lq;
  } else {
    head = (int)(r % c.n_kv);
    const long long r2 = r / c.n_kv;
    tau = (int)(r2 % total_tokens);
    layer = layer_begin + (int)(r2 / total_tokens);
  }
  int lo = 0, hi = n - 1;  // largest i with s_tok_off[i] <= tau
  while (lo < hi) {
    const int mid = (lo + hi + 1) >> 1;
    if (s_tok_off[mid] <= tau) lo = mid; else hi = mid - 1;
  }
  const int i = lo;
  const int x = s_sp[i].len + (tau - s_tok_off[i]);
  const int b = x >> c.p_log2;
  const int slot = x & (c.p - 1);
  RowUnit ru;
  if (b < s_old_nblk[i]) {
    ru.page = c.block_table[(size_t)list.ids[i] * c.max_blocks + b];
    if (!reserve && ru.page < 0) {
      // write-only call (layer_begin > 0): the slot was reserved by the layer-0 call, and an evict may
      // have run since.  A position that evict freed is dead for good - its row is not stored; any
      // other unmapped position is an error.
      SeqParams cur = s_sp[i];
      cur.len += list.n_tok[i];
      Interval dv[2];
      const int nd = dead_intervals(cur, dv);
      bool dead = false;
      for (int k = 0; k < nd; ++k) dead |= (x >= dv[k].a && x < dv[k].b);
      ru.page = dead ? kRowSkip : kRowBad;
    }
  } else if (reserve) {
    ru.page = c.free_stack[free_top - 1 - (s_blk_off[i] + (b - s_old_nblk[i]))];
  } else {
    ru.page = kRowBad;  // never read the free stack without having reserved
  }
  ru.src = (is_v ? v_new : k_new) + r * 16 + sub;
  ru.is_v = is_v;
  // pre-swizzled row (see device_state.cuh): chunk `sub` of slot `slot` sits at position sub ^ (slot & 7)
  ru.off0 = row_offset(c, layer, 0, head, slot) + (size_t)((sub ^ (slot & 7)) << 4);
  return ru;
}

// Block -> page as the eviction tasks of the fused prologue see it: blocks the append is about to
// map are not in the table yet (the commit comes after the ticket) - their pages are the ones the
// append pops, free_stack[top - (b - old_nblk)].
struct StepLookup {
  const int32_t* tab;
  const int32_t* free_stack;
  int old_nblk, top;
  __device__ __forceinline__ int operator()(int b) const { return b < old_nblk ? tab[b] : free_stack[top - (b - old_nblk)]; }
};

// Products 1 and 2 of the eviction (evict_body.cuh) for the post-append state, spread over the
// warps of ALL CTAs; they read only state that nothing rewrites before the ticket.
__device__ __forceinline__ void fused_evict_tasks(const CacheView& c, const AppendList& list, int n, int free_top,
                                                  const SeqParams* s_sp, const int* s_blk_off, const int* s_old_nblk) {
  const int warp = threadIdx.x >> 5, n_warps = blockDim.x >> 5;
  for (int task = (int)blockIdx.x + (int)gridDim.x * warp; task < 2 * n; task += (int)gridDim.x * n_warps) {
    const int role = 1 + task / n, i = task % n;
    SeqParams sp = s_sp[i];
    sp.len += list.n_tok[i];
    const StepLookup lk{c.block_table + (size_t)list.ids[i] * c.max_blocks, c.free_stack, s_old_nblk[i],
                        free_top - 1 - s_blk_off[i]};
    evict_task(c, list.ids[i], sp, role, lk);
  }
}

__global__ void __launch_bounds__(kAppendThreads)
append_kernel(const __grid_constant__ CacheView c, const __grid_constant__ AppendList list, int total_tokens,
              const uint4* __restrict__ k_new, const uint4* __restrict__ v_new, int layer_begin, int n_layers_call,
              int reserve, int fuse_evict) {
  __shared__ int s_tok_off[kMaxSeqsPerLaunch + 1];
  __shared__ int s_blk_off[kMaxSeqsPerLaunch + 1];
  __shared__ int s_old_nblk[kMaxSeqsPerLaunch];
  __shared__ int s_ndead[kMaxSeqsPerLaunch];
  __shared__ int s_off[kMaxSeqsPerLaunch + 1];
  __shared__ SeqParams s_sp[kMaxSeqsPerLaunch];  // .len = fill level BEFORE this call's tokens
  __shared__ int s_flag;
  const int tid = threadIdx.x, n_threads = blockDim.x;
  const int n = list.n;
  pdl_launch_dependents();
  pdl_wait();  // the previous kernel may still be reading the tables this one rewrites
  if (blockIdx.x == 0 && tid == 0) step_stamp(c, 0);
#ifdef MURMUR_TRACE
  const unsigned long long t_wait = globaltimer_ns();
#endif
  const int free_top = c.ctrl[kCtrlFreeTop];

  // Phase A: per-sequence old fill level and new-block demand (same result in every CTA).
  for (int i = tid; i < n; i += n_threads) {
    const SeqDev& s = c.seqs[list.ids[i]];
    SeqParams sp = load_params(s);
    if (!reserve) sp.len -= list.n_tok[i];
    if (!s.active || sp.len < 0) set_error(c, 2);
    s_sp[i] = sp;
    // reserve: blocks mapped before this call.  Write-only call: every target block was mapped by the
    // reserving call, so ALL lookups go through the table (blocks at the current length).
    const int len_tab = reserve ? max(sp.len, 0) : max(sp.len, 0) + list.n_tok[i];
    s_old_nblk[i] = (len_tab + c.p - 1) >> c.p_log2;
  }
  __syncthreads();
#ifdef MURMUR_TRACE
  const unsigned long long t_ld = globaltimer_ns();
#endif
  if (tid < 32) {  // exclusive prefix sums over <= 128 sequences, in call order: 4 per lane + warp scan
    int tok4[4], blk4[4], tok = 0, blk = 0, bad = 0;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const int i = tid * 4 + k;
      tok4[k] = tok;
      blk4[k] = blk;
      if (i < n) {
        const int new_len = s_sp[i].len + list.n_tok[i];
        const int new_nblk = (new_len + c.p - 1) >> c.p_log2;
        if (new_nblk > c.max_blocks || s_sp[i].len < 0) bad = 1;
        tok += list.n_tok[i];
        blk += new_nblk - s_old_nblk[i];
      }
    }
    int tok_inc = tok, blk_inc = blk;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int t2 = __shfl_up_sync(0xffffffffu, tok_inc, o), b2 = __shfl_up_sync(0xffffffffu, blk_inc, o);
      if (tid >= o) { tok_inc += t2; blk_inc += b2; }
    }
    const int tok_ex = tok_inc - tok, blk_ex = blk_inc - blk;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const int i = tid * 4 + k;
      if (i < n) {
        s_tok_off[i] = tok_ex + tok4[k];
        s_blk_off[i] = blk_ex + blk4[k];
      }
    }
    bad = __any_sync(0xffffffffu, bad);
    const int tok_all = __shfl_sync(0xffffffffu, tok_inc, 31), blk_all = __shfl_sync(0xffffffffu, blk_inc, 31);
    if (tid == 0) {
      s_tok_off[n] = tok_all;
      s_blk_off[n] = blk_all;
      int ok = 1;
      if (bad) { set_error(c, 2); ok = 0; }
      if (reserve && blk_all > free_top) { set_error(c, 3); ok = 0; }  // all-or-nothing
      if (tok_all != total_tokens) { set_error(c, 1); ok = 0; }
      s_flag = ok;
    }
  }
  __syncthreads();
  if (!s_flag) return;
#ifdef MURMUR_TRACE
  const unsigned long long t_a = globaltimer_ns();
#endif

  // Phase B: scatter rows.  The integer state may be committed as soon as every CTA has READ what
  // it needs of the old state (page ids); the rows themselves only have to land before the kernel
  // ends.  When the whole call is one pass over the grid (a decode step), each thread therefore
  // looks its page up, the CTA takes its ticket, and the row is stored afterwards - so the last
  // CTA's commit (+ eviction) overlaps the other CTAs' stores.
  const int sub = tid & 15;
  const int units_per_cta = n_threads >> 4;
  const long long rows_src = (long long)n_layers_call * total_tokens * c.n_kv;  // per K / per V
  const long long units = 2 * rows_src;
  const long long unit_stride = (long long)gridDim.x * units_per_cta;
  const bool one_pass = units <= unit_stride;
  int bad_page = 0;
#ifdef MURMUR_TRACE
  unsigned long long t_b = 0, t_l = 0, t_t = 0;
#define MM_STAMP(v) v = globaltimer_ns()
#else
#define MM_STAMP(v)
#endif
  if (one_pass) {
    const long long u = (long long)blockIdx.x * units_per_cta + (tid >> 4);
    RowUnit ru;
    ru.page = kRowSkip;
    uint4 val = make_uint4(0u, 0u, 0u, 0u);
    if (u < units) {
      ru = locate_row(c, list, u, rows_src, total_tokens, layer_begin, n, free_top, sub, k_new, v_new, s_tok_off,
                      s_blk_off, s_old_nblk, s_sp, reserve != 0);
      val = *ru.src;
    }
    MM_STAMP(t_l);
    if (fuse_evict) {
      fused_evict_tasks(c, list, n, free_top, s_sp, s_blk_off, s_old_nblk);
      // every CTA also counts the blocks the eviction will free (the dead ranges at the new
      // lengths; nothing remaps them before the ticket), so that the last CTA can push at once
      evict_count(c, list.ids, n, s_sp, list.n_tok, s_ndead, s_old_nblk);
    }
    MM_STAMP(t_t);
    // the barrier consumes every thread's page id: all of this CTA's reads of the old state are done
    bad_page = __syncthreads_or(ru.page == kRowBad);
    MM_STAMP(t_b);
    if (reserve) {
      if (tid == 0) s_flag = (atomicAdd(&c.ctrl[kCtrlAppendTicket], 1) == (int)gridDim.x - 1);
      __syncthreads();
    }
    if (u < units && ru.page >= 0) *ru.dst(c) = val;
  } else {
    // four rows in flight per half-warp: all page lookups and source loads first, then the stores
    for (long long u0 = (long long)blockIdx.x * units_per_cta + (tid >> 4); u0 < units; u0 += 4 * unit_stride) {
      RowUnit ru[4];
      uint4 val[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const long long u = u0 + k * unit_stride;
        ru[k].page = kRowSkip;  // no row
        if (u < units) {
          ru[k] = locate_row(c, list, u, rows_src, total_tokens, layer_begin, n, free_top, sub, k_new, v_new, s_tok_off,
                             s_blk_off, s_old_nblk, s_sp, reserve != 0);
          val[k] = *ru[k].src;
        }
      }
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        if (ru[k].page >= 0) *ru[k].dst(c) = val[k];
        else if (ru[k].page == kRowBad) bad_page = 1;
      }
    }
    if (fuse_evict) fused_evict_tasks(c, list, n, free_top, s_sp, s_blk_off, s_old_nblk);
    bad_page = __syncthreads_or(bad_page);  // every store above has consumed its page id
    if (reserve) {
      if (tid == 0) s_flag = (atomicAdd(&c.ctrl[kCtrlAppendTicket], 1) == (int)gridDim.x - 1);
      __syncthreads();
    }
  }
  if (bad_page && tid == 0) set_error(c, 2);
  if (!reserve || !s_flag) return;
#ifdef MURMUR_TRACE
  if (tid == 0) {
    unsigned long long* tr = c.timeline + (size_t)kMaxAttnGrid * kTimelineWords;
    tr[5] = t_wait; tr[6] = t_ld; tr[7] = t_a; tr[8] = t_l; tr[9] = t_t; tr[10] = t_b; tr[11] = blockIdx.x;
  }
#endif

  // Phase C: the last CTA through the ticket commits the new integer state.
  if (tid == 0) step_stamp(c, 1);
  for (int i = tid; i < n; i += n_threads) {
    SeqDev& s = c.seqs[list.ids[i]];
    const int new_len = s_sp[i].len + list.n_tok[i];
    const int new_nblk = (new_len + c.p - 1) >> c.p_log2;
    int32_t* tab = c.block_table + (size_t)list.ids[i] * c.max_blocks;
    for (int b = s_old_nblk[i]; b < new_nblk; ++b)
      tab[b] = c.free_stack[free_top - 1 - (s_blk_off[i] + (b - s_old_nblk[i]))];
    s.len = new_len;
    s_sp[i].len = new_len;
  }
  const int free_top_new = free_top - s_blk_off[n];
  if (tid == 0) {
    c.ctrl[kCtrlFreeTop] = free_top_new;
    c.ctrl[kCtrlAppendTicket] = 0;
    step_stamp(c, 2);
  }
  if (!fuse_evict) return;
  __syncthreads();  // the committed lengths and table entries, CTA-wide
  if (tid == 0) step_stamp(c, 3);
  evict_free(c, list.ids, n, s_sp, free_top_new, s_ndead, s_off, /*counted=*/one_pass);
  if (tid == 0) step_stamp(c, 4);
}

// ---- introspection helpers ------------------------------------------------------------------------
__global__ void expand_retained_kernel(CacheView c, int seq, int32_t* __restrict__ out, int cap) {
  const SeqDev& s = c.seqs[seq];
  int off = 0;
  for (int r = 0; r < s.n_runs; ++r) {
    const int first = s.runs[r][0], n = s.runs[r][1];
    for (int k = threadIdx.x; k < n; k += blockDim.x)
      if (off + k < cap) out[off + k] = first + k;
    off += n;
  }
}

__global__ void gather_kernel(CacheView c, int seq, const int32_t* __restrict__ pos, int n, int layer_begin,
                              int n_layers_call, uint4* __restrict__ k_out, uint4* __restrict__ v_out) {
  const int sub = threadIdx.x & 15;
  const long long rows = (long long)n_layers_call * n * c.n_kv;
  const long long stride = (long long)gridDim.x * (blockDim.x / 16);
  for (long long u = (long long)blockIdx.x * (blockDim.x / 16) + (threadIdx.x >> 4); u < 2 * rows; u += stride) {
    const int is_v = u >= rows;
    const long long r = is_v ? u - rows : u;
    const int head = (int)(r % c.n_kv);
    const long long r2 = r / c.n_kv;
    const int j = (int)(r2 % n);
    const int layer = layer_begin + (int)(r2 / n);
    const int x = pos[j];
    const int page = (x >= 0 && (x >> c.p_log2) < c.max_blocks)
                         ? c.block_table[(size_t)seq * c.max_blocks + (x >> c.p_log2)] : -1;
    uint4 val = make_uint4(0, 0, 0, 0);
    if (page >= 0) {
      const int slot = x & (c.p - 1);
      const uint8_t* pool = reinterpret_cast<const uint8_t*>(is_v ? c.v_pool : c.k_pool);
      val = reinterpret_cast<const uint4*>(pool + row_offset(c, layer, page, head, slot))[sub ^ (slot & 7)];
    } else if (sub == 0) {
      set_error(c, 2);
    }
    (is_v ? v_out : k_out)[r * 16 + sub] = val;
  }
}

}  // namespace

cudaError_t launch_init(const CacheView& c, cudaStream_t st, LaunchInfo* info) {
  const int n_counters = c.n_layers * kMaxSeqsPerLaunch * c.n_kv;
  init_kernel<<<256, 256, 0, st>>>(c, n_counters);
  info->launches += 1;
  return cudaGetLastError();
}

cudaError_t launch_seq_begin(const CacheView& c, int seq, const SeqParams& sp, cudaStream_t st, LaunchInfo* info) {
  seq_begin_kernel<<<1, 256, 0, st>>>(c, seq, sp);
  info->launches += 1;
  return cudaGetLastError();
}

cudaError_t launch_seq_end(const CacheView& c, int seq, cudaStream_t st, LaunchInfo* info) {
  seq_end_kernel<<<1, 32, 0, st>>>(c, seq);
  info->launches += 1;
  return cudaGetLastError();
}

cudaError_t launch_append(const CacheView& c, const AppendList& list, int total_tokens, const void* k_new,
                          const void* v_new, int layer_begin, int layer_end, bool reserve, bool fuse_evict,
                          int sm_count, bool pdl, cudaStream_t st, LaunchInfo* info) {
  const int n_layers_call = layer_end - layer_begin;
  const long long units = 2LL * n_layers_call * total_tokens * c.n_kv;
  const bool fused = reserve && fuse_evict;
  const int threads = kAppendThreads;
  long long grid = (units + (threads / 16) - 1) / (threads / 16);
  const long long cap = (long long)sm_count * (2048 / threads);
  if (grid > cap) grid = cap;
  if (grid < 1) grid = 1;
  PdlLaunch l(dim3((unsigned)grid), dim3((unsigned)threads), 0, st, pdl);
  info->launches += 1;
  info->grid = (int)grid;
  return cudaLaunchKernelEx(&l.cfg, append_kernel, c, list, total_tokens, reinterpret_cast<const uint4*>(k_new),
                            reinterpret_cast<const uint4*>(v_new), layer_begin, n_layers_call, reserve ? 1 : 0,
                            fused ? 1 : 0);
}

cudaError_t launch_expand_retained(const CacheView& c, int seq, int32_t* pos_out_dev, int cap, cudaStream_t st,
                                   LaunchInfo* info) {
  expand_retained_kernel<<<1, 256, 0, st>>>(c, seq, pos_out_dev, cap);
  info->launches += 1;
  return cudaGetLastError();
}

cudaError_t launch_gather(const CacheView& c, int seq, const int32_t* positions_dev, int n, int layer_begin,
                          int layer_end, void* k_out, void* v_out, cudaStream_t st, LaunchInfo* info) {
  const int n_layers_call = layer_end - layer_begin;
  const long long units = 2LL * n_layers_call * n * c.n_kv;
  long long grid = (units + 15) / 16;
  if (grid > 4096) grid = 4096;
  if (grid < 1) grid = 1;
  gather_kernel<<<(int)grid, 256, 0, st>>>(c, seq, positions_dev, n, layer_begin, n_layers_call,
                                           reinterpret_cast<uint4*>(k_out), reinterpret_cast<uint4*>(v_out));
  info->launches += 1;
  return cudaGetLastError();
}

}  // namespace murmur
