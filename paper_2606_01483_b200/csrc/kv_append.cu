// murmur_kv_append and the small state kernels (init, seq_begin, seq_end, gather, expand).
//
// append (the cache C receives the K,V of decode step j; prefill uses the
// same call): ONE kernel.  Every CTA recomputes the (tiny) page allocation of the call from
// the old device state - an exclusive prefix sum of per-sequence new-block counts, pages popped
// from the top of the free stack in call order (C3) - scatters its share of the rows
// into the pre-swizzled pools, and the LAST CTA to finish (ticket counter) commits the new
// lengths, block-table entries and free-stack height.  No host sync, graph-capturable.
#include "device_state.cuh"

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
constexpr int kAppendThreads = 256;

__global__ void __launch_bounds__(kAppendThreads)
append_kernel(CacheView c, AppendList list, int total_tokens, const uint4* __restrict__ k_new,
              const uint4* __restrict__ v_new, int layer_begin, int n_layers_call, int reserve) {
  __shared__ int s_tok_off[kMaxSeqsPerLaunch + 1];
  __shared__ int s_blk_off[kMaxSeqsPerLaunch + 1];
  __shared__ int s_old_len[kMaxSeqsPerLaunch];
  __shared__ int s_old_nblk[kMaxSeqsPerLaunch];
  __shared__ int s_flag;
  const int tid = threadIdx.x;
  const int n = list.n;
  const int free_top = c.ctrl[kCtrlFreeTop];

  // Phase A: per-sequence old fill level and new-block demand (same result in every CTA).
  if (tid < n) {
    const SeqDev& s = c.seqs[list.ids[tid]];
    const int old_len = reserve ? s.len : s.len - list.n_tok[tid];
    s_old_len[tid] = old_len;
    s_old_nblk[tid] = (old_len + c.p - 1) >> c.p_log2;
    if (!s.active || old_len < 0) set_error(c, 2);
  }
  __syncthreads();
  if (tid == 0) {  // exclusive prefix sums over <= 128 sequences, in call order
    int tok = 0, blk = 0, bad = 0;
    for (int i = 0; i < n; ++i) {
      s_tok_off[i] = tok;
      s_blk_off[i] = blk;
      const int new_len = s_old_len[i] + list.n_tok[i];
      const int new_nblk = (new_len + c.p - 1) >> c.p_log2;
      if (new_nblk > c.max_blocks) bad = 1;
      tok += list.n_tok[i];
      blk += new_nblk - s_old_nblk[i];
    }
    s_tok_off[n] = tok;
    s_blk_off[n] = blk;
    int ok = 1;
    if (bad) { set_error(c, 2); ok = 0; }
    if (reserve && blk > free_top) { set_error(c, 3); ok = 0; }  // all-or-nothing
    if (tok != total_tokens) { set_error(c, 1); ok = 0; }
    s_flag = ok;
  }
  __syncthreads();
  if (!s_flag) return;

  // Phase B: scatter rows.  One half-warp moves one 256-byte row (16 lanes x 16 bytes).
  const int sub = tid & 15;
  const long long rows_src = (long long)n_layers_call * total_tokens * c.n_kv;  // per K / per V
  const long long units = 2 * rows_src;
  const long long unit_stride = (long long)gridDim.x * (kAppendThreads / 16);
  for (long long u = (long long)blockIdx.x * (kAppendThreads / 16) + (tid >> 4); u < units; u += unit_stride) {
    const int is_v = u >= rows_src;
    const long long r = is_v ? u - rows_src : u;
    const int head = (int)(r % c.n_kv);
    const long long r2 = r / c.n_kv;
    const int tau = (int)(r2 % total_tokens);
    const int layer = layer_begin + (int)(r2 / total_tokens);
    int lo = 0, hi = n - 1;  // largest i with s_tok_off[i] <= tau
    while (lo < hi) {
      const int mid = (lo + hi + 1) >> 1;
      if (s_tok_off[mid] <= tau) lo = mid; else hi = mid - 1;
    }
    const int i = lo;
    const int x = s_old_len[i] + (tau - s_tok_off[i]);
    const int b = x >> c.p_log2;
    const int slot = x & (c.p - 1);
    int page;
    if (b < s_old_nblk[i]) page = c.block_table[(size_t)list.ids[i] * c.max_blocks + b];
    else page = c.free_stack[free_top - 1 - (s_blk_off[i] + (b - s_old_nblk[i]))];
    const uint4 val = (is_v ? v_new : k_new)[r * 16 + sub];
    uint8_t* pool = reinterpret_cast<uint8_t*>(is_v ? c.v_pool : c.k_pool);
    uint4* dst = reinterpret_cast<uint4*>(pool + row_offset(c, layer, page, head, slot));
    dst[sub ^ (slot & 7)] = val;  // pre-swizzled row (see device_state.cuh)
  }
  if (!reserve) return;

  // Phase C: the last CTA to finish commits the new integer state.
  __threadfence();
  __syncthreads();
  if (tid == 0) s_flag = (atomicAdd(&c.ctrl[kCtrlAppendTicket], 1) == (int)gridDim.x - 1);
  __syncthreads();
  if (!s_flag) return;
  __threadfence();
  for (int i = tid; i < n; i += kAppendThreads) {
    SeqDev& s = c.seqs[list.ids[i]];
    const int new_len = s_old_len[i] + list.n_tok[i];
    const int new_nblk = (new_len + c.p - 1) >> c.p_log2;
    int32_t* tab = c.block_table + (size_t)list.ids[i] * c.max_blocks;
    for (int b = s_old_nblk[i]; b < new_nblk; ++b)
      tab[b] = c.free_stack[free_top - 1 - (s_blk_off[i] + (b - s_old_nblk[i]))];
    s.len = new_len;
  }
  if (tid == 0) {
    c.ctrl[kCtrlFreeTop] = free_top - s_blk_off[n];
    c.ctrl[kCtrlAppendTicket] = 0;
  }
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
                          const void* v_new, int layer_begin, int layer_end, bool reserve, int sm_count,
                          cudaStream_t st, LaunchInfo* info) {
  const int n_layers_call = layer_end - layer_begin;
  const long long units = 2LL * n_layers_call * total_tokens * c.n_kv;
  long long grid = (units + (kAppendThreads / 16) - 1) / (kAppendThreads / 16);
  const long long cap = (long long)sm_count * 8;
  if (grid > cap) grid = cap;
  if (grid < 1) grid = 1;
  append_kernel<<<(int)grid, kAppendThreads, 0, st>>>(c, list, total_tokens, reinterpret_cast<const uint4*>(k_new),
                                                      reinterpret_cast<const uint4*>(v_new), layer_begin,
                                                      n_layers_call, reserve ? 1 : 0);
  info->launches += 1;
  info->grid = (int)grid;
  return cudaGetLastError();
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
