// Host side of the C ABI (include/murmur.h): handle, workspace carve-up, argument validation
// against a host mirror of the integer state, kernel dispatch, introspection.
//
// The mirror holds, per sequence, only (regions, policy, length, length at the last evict, blocks
// freed so far); with the closed form in policy_math.cuh that is enough to know the free-page
// count exactly, so page exhaustion is reported synchronously and all-or-nothing without ever
// reading device memory.  Every state transition itself runs in the kernels.
#include <cuda_runtime.h>

#include <atomic>
#include <cstring>
#include <new>
#include <vector>

#include "../../include/murmur.h"
#include "device_state.cuh"

using namespace murmur;

namespace murmur {
cudaError_t opt_in_smem_once(int slot, const void* func, int smem) {
  constexpr int kMaxDevices = 64;
  static std::atomic<bool> done[kSmemKernels][kMaxDevices];  // zero-initialised; setting twice is harmless
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  const bool tracked = slot >= 0 && slot < kSmemKernels && dev >= 0 && dev < kMaxDevices;
  if (tracked && done[slot][dev].load(std::memory_order_acquire)) return cudaSuccess;
  e = cudaFuncSetAttribute(func, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
  if (e == cudaSuccess && tracked) done[slot][dev].store(true, std::memory_order_release);
  return e;
}
}  // namespace murmur

namespace {

struct HostSeq {
  bool active = false;
  SeqParams sp{};
  int32_t evict_len = -1;   // length when murmur_kv_evict last ran (-1: never)
  int32_t freed_blocks = 0;  // blocks of this sequence returned to the pool so far
  bool indexed = false;      // indexed mode (kv_indexed.cu): the positional fields above are frozen
  int32_t idx_blocks = 0;    // blocks mapped in indexed mode
  int32_t idx_max_len = 0;   // rows of the longest slab
  // Open decode step (murmur_decode_step_layers): the length the opening call left the sequence at, and the layers
  // whose range has not been issued yet (bit l).  open_len == -1: no step is open.
  // (Fixed-size bitmap: layers >= 256 are counted but a repeated issue of one of them is not detected.)
  int32_t open_len = -1;
  int32_t open_left = 0;  // layers not issued yet
  uint64_t open_todo[4] = {0, 0, 0, 0};
};

constexpr size_t kAlign = 256;
inline size_t align_up(size_t x) { return (x + kAlign - 1) / kAlign * kAlign; }

struct Carve {
  size_t seqs, block_table, live_pages, live_blocks, tiles, free_stack, ctrl, counters, partials, timeline;
  size_t stage_k, stage_v, stage_q, stage_out, scratch;
  size_t total;
  int stage_seqs;
  size_t scratch_ints;
};

bool geometry_ok(const murmur_cache_desc_t* d) {
  if (!d) return false;
  if (d->head_dim != kHeadDim) return false;
  if (d->n_layers < 1 || d->n_kv_heads < 1 || d->n_q_heads < 1) return false;
  if (d->n_q_heads % d->n_kv_heads) return false;
  if (d->n_q_heads / d->n_kv_heads > kMaxGroup) return false;
  if (d->page_size < 1 || d->page_size > kTileRows || (d->page_size & (d->page_size - 1))) return false;
  if (d->max_seqs < 1 || d->max_blocks_per_seq < 1 || d->n_pages < 1) return false;
  if (d->n_pages > 0x7fffffffLL) return false;
  if ((int64_t)d->max_blocks_per_seq * d->page_size > 0x7fffffffLL) return false;
  return true;
}

Carve carve(const murmur_cache_desc_t* d) {
  Carve c{};
  size_t off = 0;
  auto take = [&](size_t bytes) {
    const size_t at = off;
    off = align_up(off + bytes);
    return at;
  };
  const size_t tab = (size_t)d->max_seqs * d->max_blocks_per_seq;
  c.seqs = take((size_t)d->max_seqs * sizeof(SeqDev));
  c.block_table = take(tab * 4);
  c.live_pages = take(tab * 4);
  c.live_blocks = take(tab * 4);
  c.tiles = take(tab * sizeof(TileDesc));
  c.free_stack = take((size_t)d->n_pages * 4);
  c.ctrl = take(kCtrlWords * 4);
  c.counters = take((size_t)d->n_layers * kMaxSeqsPerLaunch * d->n_kv_heads * 4);
  c.partials = take((size_t)4 * kMaxAttnGrid * kPartialFloats * 4);
  c.timeline = take(((size_t)kMaxAttnGrid * kTimelineWords + kStepTraceWords) * 8);
  c.stage_seqs = d->max_seqs < kMaxSeqsPerLaunch ? d->max_seqs : kMaxSeqsPerLaunch;
  const size_t kv_b = (size_t)d->n_layers * c.stage_seqs * d->n_kv_heads * kRowBytes;
  const size_t q_b = (size_t)d->n_layers * c.stage_seqs * d->n_q_heads * kRowBytes;
  c.stage_k = take(kv_b);
  c.stage_v = take(kv_b);
  c.stage_q = take(q_b);
  c.stage_out = take(q_b);
  c.scratch_ints = (size_t)d->max_blocks_per_seq * d->page_size;
  c.scratch = take(c.scratch_ints * 4);
  c.total = off;
  return c;
}

}  // namespace

struct murmur_cache {
  murmur_cache_desc_t desc;
  CacheView view;
  Carve cv;
  std::vector<HostSeq> seqs;
  int64_t free_pages;
  int sm_count;
  int l2_bytes = 0;
  int attn_variant_opt;
  int attn_grid_opt;
  int pdl_opt;         // programmatic dependent launch between the kernels of a step
  int fuse_step_opt;   // murmur_decode_step: append + evict in one launch
  int prefill_variant_opt;  // MURMUR_PREFILL_*
  int host_zero_copy_opt;   // murmur_decode_step_host: work on page-locked host buffers in place
  int l2_keep_pct_opt;      // MURMUR_OPT_L2_KEEP_PCT (-1 = automatic)
  murmur_stats_t stats;
  cudaError_t last_cuda;
  uint8_t* ws;
  bool chain_ok = false;        // the last launch through this handle was a (counted) step launch: the next may chain
  uint32_t step_done = 0;       // value kCtrlStepDone reaches once every step launch counted so far is through its keepers
  IdxView idx{nullptr, nullptr, 0};        // indexed-mode tables (murmur_indexed_enable)
  unsigned long long* idx_moved = nullptr;  // device counter of rows moved by the last index-set eviction
  // A call was recorded into a CUDA graph: the host mirror (lengths, free pages, open steps) was advanced although
  // nothing ran, and replays will advance the device without the mirror.  Until murmur_mirror_sync has re-read the
  // device state, every state-dependent call outside a capture returns MURMUR_ERR_STATE.
  bool mirror_stale = false;
};

namespace {

murmur_status_t cuda_fail(murmur_cache* c, cudaError_t e) {
  c->last_cuda = e;
  return MURMUR_ERR_CUDA;
}

#define MM_CUDA(c, expr)                                  \
  do {                                                    \
    cudaError_t e__ = (expr);                             \
    if (e__ != cudaSuccess) return cuda_fail((c), e__);   \
  } while (0)

void note(murmur_cache* c, const LaunchInfo& li) {
  c->stats.kernel_launches += li.launches;
  c->chain_ok = false;  // any launch that is not a step launch breaks the chain (the step path sets it again)
}

inline int32_t blocks_for(int32_t len, int32_t p) { return (len + p - 1) / p; }

// ids in range, active, distinct; want_indexed: 0 = positional sequences only, 1 = indexed-mode sequences only
// Fraction of the K/V rows a decode-attention launch reads with L2::evict_last (MURMUR_OPT_L2_KEEP_PCT).  The default
// is 0: a pure evict_first stream that leaves the L2 to whatever else the engine runs between two attention calls
// (its GEMMs and activations) - lines marked evict_last are never demoted by this library, and a benchmark of
// back-to-back attention steps cannot see what they cost the neighbours.  Opt-in, -1 = automatic: consecutive steps
// re-read the same retained rows (the windows move by one token), so when the retained rows of the sequences IN THE
// CALL, over all layers, are not much more than the L2 holds, half an L2 of them is pinned ahead of the rest and
// served from there on the next step (config 3b, 151 MB per step: 29.8 -> 26.9 us).  For larger working sets any
// pinned share measured slower than a pure evict_first stream (config 2, 575 MB: 89 -> 92-97 us), so they get none.
constexpr double kL2KeepShare = 0.5, kL2KeepMaxWorkingSet = 1.3;  // in units of the L2 size
float l2_keep_fraction(murmur_cache* c, const int32_t* seq_ids, int32_t n_seqs) {
  if (c->l2_keep_pct_opt >= 0) return (float)c->l2_keep_pct_opt / 100.f;
  double rows = 0;
  for (int i = 0; i < n_seqs; ++i) rows += (double)retained_count(c->seqs[seq_ids[i]].sp);
  const double bytes = rows * 2.0 * kRowBytes * c->desc.n_kv_heads * c->desc.n_layers;
  if (bytes <= 0 || bytes > kL2KeepMaxWorkingSet * (double)c->l2_bytes) return 0.f;
  const double f = kL2KeepShare * (double)c->l2_bytes / bytes;
  return (float)(f > 1.0 ? 1.0 : f);
}

// First line of every call that reads or advances the host mirror.  While `stream` is being captured the call is
// let through and the handle is marked; afterwards calls are refused until murmur_mirror_sync has run.
murmur_status_t mirror_guard(murmur_cache* c, void* stream) {
  cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
  if (cudaStreamIsCapturing((cudaStream_t)stream, &cap) == cudaSuccess && cap != cudaStreamCaptureStatusNone) {
    c->mirror_stale = true;
    return MURMUR_OK;
  }
  return c->mirror_stale ? MURMUR_ERR_STATE : MURMUR_OK;
}
#define MM_GUARD(c, stream)                                   \
  do {                                                        \
    if ((c) != nullptr) {                                     \
      murmur_status_t g__ = mirror_guard((c), (stream));      \
      if (g__ != MURMUR_OK) return g__;                       \
    }                                                         \
  } while (0)

// ---- open-step bookkeeping (murmur_decode_step_layers) ----
void open_step_mark(murmur_cache* c, HostSeq& hs, int32_t layer_begin, int32_t layer_end, bool opens) {
  const int L = c->desc.n_layers;
  if (opens) {
    hs.open_len = hs.sp.len;
    hs.open_left = L;
    for (int w = 0; w < 4; ++w) hs.open_todo[w] = 0;
    for (int l = 0; l < L && l < 256; ++l) hs.open_todo[l >> 6] |= 1ull << (l & 63);
  }
  for (int l = layer_begin; l < layer_end; ++l) {
    if (l < 256) hs.open_todo[l >> 6] &= ~(1ull << (l & 63));
    hs.open_left -= 1;
  }
  if (hs.open_left <= 0) hs.open_len = -1;  // every layer issued: the step is closed
}
bool open_step_has(const HostSeq& hs, int32_t layer_begin, int32_t layer_end) {
  if (hs.open_len < 1 || hs.open_len != hs.sp.len || hs.evict_len != hs.sp.len) return false;
  for (int l = layer_begin; l < layer_end && l < 256; ++l)
    if (!((hs.open_todo[l >> 6] >> (l & 63)) & 1ull)) return false;
  return true;
}

murmur_status_t check_ids(murmur_cache* c, const int32_t* ids, int32_t n, int want_indexed = 0) {
  if (!ids || n < 0) return MURMUR_ERR_INVALID_ARG;
  for (int i = 0; i < n; ++i) {
    if (ids[i] < 0 || ids[i] >= c->desc.max_seqs) return MURMUR_ERR_INVALID_ARG;
    for (int j = 0; j < i; ++j)
      if (ids[j] == ids[i]) return MURMUR_ERR_INVALID_ARG;
  }
  for (int i = 0; i < n; ++i)
    if (!c->seqs[ids[i]].active || (int)c->seqs[ids[i]].indexed != want_indexed) return MURMUR_ERR_STATE;
  return MURMUR_OK;
}

}  // namespace

extern "C" {

static murmur_status_t check_seq(murmur_cache_t* c, int32_t seq);

size_t murmur_pool_bytes(const murmur_cache_desc_t* d) {
  if (!geometry_ok(d)) return 0;
  return (size_t)d->n_layers * (size_t)d->n_pages * d->n_kv_heads * d->page_size * kRowBytes;
}

size_t murmur_workspace_bytes(const murmur_cache_desc_t* d) {
  if (!geometry_ok(d)) return 0;
  return carve(d).total;
}

murmur_status_t murmur_cache_create(const murmur_cache_desc_t* d, murmur_cache_t** out, void* stream) {
  if (!d || !out) return MURMUR_ERR_INVALID_ARG;
  if (!geometry_ok(d)) return MURMUR_ERR_UNSUPPORTED;
  if (!d->k_pool || !d->v_pool || !d->workspace) return MURMUR_ERR_INVALID_ARG;
  if (((uintptr_t)d->k_pool | (uintptr_t)d->v_pool | (uintptr_t)d->workspace) & (kAlign - 1)) return MURMUR_ERR_INVALID_ARG;
  const Carve cv = carve(d);
  if (d->workspace_bytes < cv.total) return MURMUR_ERR_INVALID_ARG;
  murmur_cache* c = new (std::nothrow) murmur_cache();
  if (!c) return MURMUR_ERR_INVALID_ARG;
  c->desc = *d;
  c->cv = cv;
  c->ws = reinterpret_cast<uint8_t*>(d->workspace);
  c->seqs.assign(d->max_seqs, HostSeq());
  c->free_pages = d->n_pages;
  c->attn_variant_opt = MURMUR_ATTN_AUTO;
  c->attn_grid_opt = 0;
  c->pdl_opt = 1;
  c->fuse_step_opt = 2;
  c->prefill_variant_opt = MURMUR_PREFILL_AUTO;
  c->host_zero_copy_opt = 1;
  c->l2_keep_pct_opt = 0;
  std::memset(&c->stats, 0, sizeof c->stats);
  c->last_cuda = cudaSuccess;
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, dev);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&c->l2_bytes, cudaDevAttrL2CacheSize, dev);
  if (e != cudaSuccess) {
    delete c;
    return MURMUR_ERR_CUDA;
  }
  CacheView& v = c->view;
  v.n_layers = d->n_layers; v.n_q = d->n_q_heads; v.n_kv = d->n_kv_heads;
  v.p = d->page_size;
  v.p_log2 = 0;
  while ((1 << v.p_log2) < d->page_size) ++v.p_log2;
  v.max_seqs = d->max_seqs; v.max_blocks = d->max_blocks_per_seq;
  v.group = d->n_q_heads / d->n_kv_heads;
  v.n_pages = d->n_pages;
  v.k_pool = reinterpret_cast<uint16_t*>(d->k_pool);
  v.v_pool = reinterpret_cast<uint16_t*>(d->v_pool);
  v.seqs = reinterpret_cast<SeqDev*>(c->ws + cv.seqs);
  v.block_table = reinterpret_cast<int32_t*>(c->ws + cv.block_table);
  v.live_pages = reinterpret_cast<int32_t*>(c->ws + cv.live_pages);
  v.live_blocks = reinterpret_cast<int32_t*>(c->ws + cv.live_blocks);
  v.tiles = reinterpret_cast<TileDesc*>(c->ws + cv.tiles);
  v.free_stack = reinterpret_cast<int32_t*>(c->ws + cv.free_stack);
  v.ctrl = reinterpret_cast<int32_t*>(c->ws + cv.ctrl);
  v.item_counters = reinterpret_cast<int32_t*>(c->ws + cv.counters);
  v.partials = reinterpret_cast<float*>(c->ws + cv.partials);
  v.timeline = reinterpret_cast<unsigned long long*>(c->ws + cv.timeline);
  LaunchInfo li{};
  e = launch_init(v, (cudaStream_t)stream, &li);
  if (e != cudaSuccess) {
    delete c;
    return MURMUR_ERR_CUDA;
  }
  note(c, li);
  c->stats.sm_count = c->sm_count;
  c->stats.free_pages = c->free_pages;
  *out = c;
  return MURMUR_OK;
}

murmur_status_t murmur_cache_destroy(murmur_cache_t* c) {
  delete c;
  return MURMUR_OK;
}

murmur_status_t murmur_seq_begin(murmur_cache_t* c, int32_t seq, int32_t n_prefix, int32_t n_speech, int32_t n_mid,
                                 const murmur_policy_t* pol, void* stream) {
  if (!c || !pol) return MURMUR_ERR_INVALID_ARG;
  MM_GUARD(c, stream);
  if (seq < 0 || seq >= c->desc.max_seqs) return MURMUR_ERR_INVALID_ARG;
  if (n_prefix < 0 || n_speech < 0 || n_mid < 0) return MURMUR_ERR_INVALID_ARG;
  if (pol->w_speech < 0 || pol->delay < 0 || pol->n_sink_speech < 0 || pol->w_out < 0 || pol->n_sink_out < 0)
    return MURMUR_ERR_INVALID_ARG;
  if ((int64_t)n_prefix + n_speech + n_mid > (int64_t)c->desc.max_blocks_per_seq * c->desc.page_size)
    return MURMUR_ERR_INVALID_ARG;
  HostSeq& hs = c->seqs[seq];
  if (hs.active) return MURMUR_ERR_STATE;
  SeqParams sp{};
  sp.P = n_prefix; sp.S = n_speech; sp.M = n_mid; sp.len = 0;
  sp.w_s = pol->w_speech; sp.d = pol->delay; sp.k_s = pol->n_sink_speech;
  sp.w_o = pol->w_out; sp.k_o = pol->n_sink_out;
  LaunchInfo li{};
  MM_CUDA(c, launch_seq_begin(c->view, seq, sp, (cudaStream_t)stream, &li));
  note(c, li);
  hs = HostSeq();
  hs.active = true;
  hs.sp = sp;
  return MURMUR_OK;
}

murmur_status_t murmur_seq_end(murmur_cache_t* c, int32_t seq, void* stream) {
  if (!c) return MURMUR_ERR_INVALID_ARG;
  MM_GUARD(c, stream);
  if (seq < 0 || seq >= c->desc.max_seqs) return MURMUR_ERR_INVALID_ARG;
  HostSeq& hs = c->seqs[seq];
  if (!hs.active) return MURMUR_ERR_STATE;
  LaunchInfo li{};
  if (hs.indexed) {
    MM_CUDA(c, launch_indexed_seq_end(c->view, seq, (cudaStream_t)stream, &li));
    note(c, li);
    c->free_pages += hs.idx_blocks;
    c->stats.free_pages = c->free_pages;
    hs = HostSeq();
    return MURMUR_OK;
  }
  MM_CUDA(c, launch_seq_end(c->view, seq, (cudaStream_t)stream, &li));
  note(c, li);
  c->free_pages += blocks_for(hs.sp.len, c->desc.page_size) - hs.freed_blocks;
  c->stats.free_pages = c->free_pages;
  hs = HostSeq();
  return MURMUR_OK;
}

// Host mirror of what an evict at the sequences' current lengths frees (closed form).
static void mirror_evict(murmur_cache_t* c, const int32_t* seq_ids, int32_t n_seqs) {
  for (int i = 0; i < n_seqs; ++i) {
    HostSeq& hs = c->seqs[seq_ids[i]];
    const int32_t dead = dead_block_count(hs.sp, c->desc.page_size);
    c->free_pages += dead - hs.freed_blocks;
    hs.freed_blocks = dead;
    hs.evict_len = hs.sp.len;
  }
  c->stats.free_pages = c->free_pages;
  c->stats.evict_calls += 1;
}

// fuse_evict: the append kernel's last CTA also runs the eviction body for the same sequences
// (single launch of <= 128 sequences, layer_begin == 0 only).
static murmur_status_t append_impl(murmur_cache_t* c, const int32_t* seq_ids, const int32_t* n_tokens, int32_t n_seqs,
                                   const void* k_new, const void* v_new, int32_t layer_begin, int32_t layer_end,
                                   bool fuse_evict, void* stream) {
  if (!c || !n_tokens) return MURMUR_ERR_INVALID_ARG;
  MM_GUARD(c, stream);
  murmur_status_t st = check_ids(c, seq_ids, n_seqs);
  if (st != MURMUR_OK) return st;
  if (layer_begin < 0 || layer_end > c->desc.n_layers || layer_begin >= layer_end) return MURMUR_ERR_INVALID_ARG;
  const bool reserve = (layer_begin == 0);
  const int32_t p = c->desc.page_size;
  int64_t total = 0, need = 0;
  for (int i = 0; i < n_seqs; ++i) {
    if (n_tokens[i] < 0) return MURMUR_ERR_INVALID_ARG;
    const HostSeq& hs = c->seqs[seq_ids[i]];
    total += n_tokens[i];
    if (reserve) {
      const int64_t new_len = (int64_t)hs.sp.len + n_tokens[i];
      if (new_len > (int64_t)c->desc.max_blocks_per_seq * p) return MURMUR_ERR_STATE;
      need += blocks_for((int32_t)new_len, p) - blocks_for(hs.sp.len, p);
    } else if (n_tokens[i] > hs.sp.len) {
      return MURMUR_ERR_STATE;  // rows for positions that were never reserved
    }
  }
  if (total > 0x7fffffffLL) return MURMUR_ERR_INVALID_ARG;
  if (total > 0 && (!k_new || !v_new)) return MURMUR_ERR_INVALID_ARG;
  if (reserve && need > c->free_pages) return MURMUR_ERR_OOM_PAGES;  // all-or-nothing
  if (n_seqs == 0 || total == 0) return MURMUR_OK;

  // split into launches of <= 128 sequences, in call order
  const size_t row_tok = (size_t)c->desc.n_kv_heads * kRowBytes;
  int64_t tok_done = 0;
  for (int base = 0; base < n_seqs; base += kMaxSeqsPerLaunch) {
    AppendList list;
    list.n = (n_seqs - base) < kMaxSeqsPerLaunch ? (n_seqs - base) : kMaxSeqsPerLaunch;
    int64_t chunk_tok = 0;
    for (int i = 0; i < list.n; ++i) {
      list.ids[i] = seq_ids[base + i];
      list.n_tok[i] = n_tokens[base + i];
      chunk_tok += n_tokens[base + i];
    }
    if (chunk_tok > 0) {
      if (base == 0 && list.n == n_seqs) {
        LaunchInfo li{};
        MM_CUDA(c, launch_append(c->view, list, (int)chunk_tok, k_new, v_new, layer_begin, layer_end, reserve,
                                 fuse_evict, c->sm_count, c->pdl_opt != 0, (cudaStream_t)stream, &li));
        note(c, li);
      } else {
        // several chunks: the source is [layer][all tokens][...], so each layer is its own launch
        for (int layer = layer_begin; layer < layer_end; ++layer) {
          const size_t off = ((size_t)(layer - layer_begin) * (size_t)total + (size_t)tok_done) * row_tok;
          LaunchInfo li{};
          MM_CUDA(c, launch_append(c->view, list, (int)chunk_tok, (const uint8_t*)k_new + off,
                                   (const uint8_t*)v_new + off, layer, layer + 1,
                                   reserve && layer == layer_begin, false, c->sm_count, c->pdl_opt != 0,
                                   (cudaStream_t)stream, &li));
          note(c, li);
        }
      }
    }
    tok_done += chunk_tok;
  }
  if (reserve) {
    for (int i = 0; i < n_seqs; ++i) c->seqs[seq_ids[i]].sp.len += n_tokens[i];
    c->free_pages -= need;
    c->stats.free_pages = c->free_pages;
  }
  c->stats.append_calls += 1;
  if (fuse_evict) mirror_evict(c, seq_ids, n_seqs);
  return MURMUR_OK;
}

murmur_status_t murmur_kv_append(murmur_cache_t* c, const int32_t* seq_ids, const int32_t* n_tokens, int32_t n_seqs,
                                 const void* k_new, const void* v_new, int32_t layer_begin, int32_t layer_end,
                                 void* stream) {
  return append_impl(c, seq_ids, n_tokens, n_seqs, k_new, v_new, layer_begin, layer_end, false, stream);
}

murmur_status_t murmur_kv_evict(murmur_cache_t* c, const int32_t* seq_ids, int32_t n_seqs, void* stream) {
  if (!c) return MURMUR_ERR_INVALID_ARG;
  MM_GUARD(c, stream);
  murmur_status_t st = check_ids(c, seq_ids, n_seqs);
  if (st != MURMUR_OK) return st;
  for (int base = 0; base < n_seqs; base += kMaxSeqsPerLaunch) {
    SeqList list;
    list.n = (n_seqs - base) < kMaxSeqsPerLaunch ? (n_seqs - base) : kMaxSeqsPerLaunch;
    for (int i = 0; i < list.n; ++i) list.ids[i] = seq_ids[base + i];
    LaunchInfo li{};
    MM_CUDA(c, launch_evict(c->view, list, c->pdl_opt != 0, (cudaStream_t)stream, &li));
    note(c, li);
  }
  mirror_evict(c, seq_ids, n_seqs);
  return MURMUR_OK;
}

// window == nullptr: each sequence's own policy.  Otherwise the attended set is the A(t) of `window`
// (same for all listed sequences), which must lie inside what the sequence's own policy keeps resident.
static murmur_status_t attn_impl(murmur_cache_t* c, const int32_t* seq_ids, int32_t n_seqs, const void* q, void* out,
                                 float* lse, int32_t layer_begin, int32_t layer_end, float sm_scale,
                                 const murmur_policy_t* window, void* stream) {
  if (!c) return MURMUR_ERR_INVALID_ARG;
  MM_GUARD(c, stream);
  murmur_status_t st = check_ids(c, seq_ids, n_seqs);
  if (st != MURMUR_OK) return st;
  if (layer_begin < 0 || layer_end > c->desc.n_layers || layer_begin >= layer_end) return MURMUR_ERR_INVALID_ARG;
  if (!(sm_scale > 0.f)) return MURMUR_ERR_INVALID_ARG;
  if (n_seqs == 0) return MURMUR_OK;
  if (!q || !out) return MURMUR_ERR_INVALID_ARG;
  SeqParams win{};
  if (window) {
    if (window->w_speech < 0 || window->delay < 0 || window->n_sink_speech < 0 || window->w_out < 0 || window->n_sink_out < 0)
      return MURMUR_ERR_INVALID_ARG;
    win.w_s = window->w_speech; win.d = window->delay; win.k_s = window->n_sink_speech;
    win.w_o = window->w_out; win.k_o = window->n_sink_out;
  }
  for (int i = 0; i < n_seqs; ++i) {
    const HostSeq& hs = c->seqs[seq_ids[i]];
    if (hs.sp.len < 1 || hs.evict_len != hs.sp.len) return MURMUR_ERR_STATE;
    SeqParams sp = hs.sp;
    if (window) {
      // A_window(t) must avoid every position the sequence's own policy has evicted: a window that
      // trails no further back, a delay no longer, and no more sinks than the base policy's
      if (win.w_s > sp.w_s || win.d > sp.d || win.k_s > sp.k_s || win.w_o > sp.w_o || win.k_o > sp.k_o)
        return MURMUR_ERR_INVALID_ARG;
      sp.w_s = win.w_s; sp.d = win.d; sp.k_s = win.k_s; sp.w_o = win.w_o; sp.k_o = win.k_o;
    }
    if (retained_count(sp) < 1) return MURMUR_ERR_STATE;  // Eq. 1 over an empty set is undefined
  }
  int variant = c->attn_variant_opt;
  if (variant == MURMUR_ATTN_AUTO) variant = (c->desc.page_size >= 16) ? MURMUR_ATTN_MMA : MURMUR_ATTN_GENERIC;
  if (variant == MURMUR_ATTN_MMA && c->desc.page_size < 16) return MURMUR_ERR_UNSUPPORTED;
  if (window && variant != MURMUR_ATTN_MMA) return MURMUR_ERR_UNSUPPORTED;
  const int grid = c->attn_grid_opt > 0 ? c->attn_grid_opt : c->sm_count;
  const int chunk = (variant == MURMUR_ATTN_MMA) ? kMaxSeqsAttn : kMaxSeqsPerLaunch;
  for (int base = 0; base < n_seqs; base += chunk) {
    SeqList list;
    list.n = (n_seqs - base) < chunk ? (n_seqs - base) : chunk;
    for (int i = 0; i < list.n; ++i) list.ids[i] = seq_ids[base + i];
    LaunchInfo li{};
    if (variant == MURMUR_ATTN_MMA) {
      c->view.l2_keep = l2_keep_fraction(c, list.ids, list.n);
      MM_CUDA(c, launch_attn_mma(c->view, list, base, n_seqs, q, out, lse, layer_begin, layer_end, sm_scale, grid,
                                 c->pdl_opt != 0, window ? &win : nullptr, (cudaStream_t)stream, &li));
    } else {
      MM_CUDA(c, launch_attn_generic(c->view, list, base, n_seqs, q, out, lse, layer_begin, layer_end, sm_scale,
                                     (cudaStream_t)stream, &li));
    }
    note(c, li);
    c->stats.attn_grid = li.grid;
    c->stats.attn_smem_bytes = li.smem;
  }
  c->stats.attn_variant = variant;
  c->stats.attn_calls += 1;
  return MURMUR_OK;
}

murmur_status_t murmur_decode_attn(murmur_cache_t* c, const int32_t* seq_ids, int32_t n_seqs, const void* q, void* out,
                                   float* lse, int32_t layer_begin, int32_t layer_end, float sm_scale, void* stream) {
  return attn_impl(c, seq_ids, n_seqs, q, out, lse, layer_begin, layer_end, sm_scale, nullptr, stream);
}

murmur_status_t murmur_decode_attn_windowed(murmur_cache_t* c, const int32_t* seq_ids, int32_t n_seqs, const void* q,
                                            void* out, float* lse, int32_t layer_begin, int32_t layer_end,
                                            float sm_scale, const murmur_policy_t* window, void* stream) {
  if (!window) return MURMUR_ERR_INVALID_ARG;
  return attn_impl(c, seq_ids, n_seqs, q, out, lse, layer_begin, layer_end, sm_scale, window, stream);
}

// validates a 1-token-per-sequence append before anything is enqueued (all-or-nothing)
static murmur_status_t check_step(murmur_cache_t* c, const int32_t* seq_ids, int32_t n_seqs) {
  if (n_seqs < 1 || n_seqs > kMaxSeqsPerLaunch) return MURMUR_ERR_INVALID_ARG;
  murmur_status_t st = check_ids(c, seq_ids, n_seqs);
  if (st != MURMUR_OK) return st;
  int64_t need = 0;
  for (int i = 0; i < n_seqs; ++i) {
    const HostSeq& hs = c->seqs[seq_ids[i]];
    if ((int64_t)hs.sp.len + 1 > (int64_t)c->desc.max_blocks_per_seq * c->desc.page_size) return MURMUR_ERR_STATE;
    need += blocks_for(hs.sp.len + 1, c->desc.page_size) - blocks_for(hs.sp.len, c->desc.page_size);
  }
  if (need > c->free_pages) return MURMUR_ERR_OOM_PAGES;
  return MURMUR_OK;
}

// One decode step restricted to the layers [layer_begin, layer_end).  layer_begin == 0 opens the step:
// slots reserved, lengths advanced, eviction run; later ranges only write their rows and attend.
static murmur_status_t step_layers_impl(murmur_cache_t* c, const int32_t* seq_ids, int32_t n_seqs, const void* k_new,
                                        const void* v_new, const void* q, void* out, float* lse, int32_t layer_begin,
                                        int32_t layer_end, float sm_scale, void* stream) {
  if (!c || !k_new || !v_new || !q || !out) return MURMUR_ERR_INVALID_ARG;
  if (!(sm_scale > 0.f)) return MURMUR_ERR_INVALID_ARG;
  if (layer_begin < 0 || layer_end > c->desc.n_layers || layer_begin >= layer_end) return MURMUR_ERR_INVALID_ARG;
  MM_GUARD(c, stream);
  const bool opens = (layer_begin == 0);
  murmur_status_t st;
  if (opens) {
    st = check_step(c, seq_ids, n_seqs);
    if (st != MURMUR_OK) return st;
  } else {
    if (n_seqs < 1 || n_seqs > kMaxSeqsPerLaunch) return MURMUR_ERR_INVALID_ARG;
    st = check_ids(c, seq_ids, n_seqs);
    if (st != MURMUR_OK) return st;
    // the step must be open for every listed sequence (token reserved, eviction run by a layer_begin == 0 call, no
    // append or evict since) and none of these layers issued yet: a second write would overwrite the token's rows
    for (int i = 0; i < n_seqs; ++i)
      if (!open_step_has(c->seqs[seq_ids[i]], layer_begin, layer_end)) return MURMUR_ERR_STATE;
  }
  int32_t ones[kMaxSeqsPerLaunch];
  for (int i = 0; i < n_seqs; ++i) ones[i] = 1;
  int variant = c->attn_variant_opt;
  if (variant == MURMUR_ATTN_AUTO) variant = (c->desc.page_size >= 16) ? MURMUR_ATTN_MMA : MURMUR_ATTN_GENERIC;
  if (c->fuse_step_opt >= 2 && variant == MURMUR_ATTN_MMA && c->desc.page_size >= 16 && n_seqs <= kMaxSeqsAttn) {
    // ONE launch: every CTA derives the post-append state, keeper warps scatter / commit / evict
    SeqList list;
    list.n = n_seqs;
    for (int i = 0; i < n_seqs; ++i) list.ids[i] = seq_ids[i];
    const int grid = c->attn_grid_opt > 0 ? c->attn_grid_opt : c->sm_count;
    LaunchInfo li{};
    // chained steps (decode_attn_mma.cu): only between launches the host has counted - not while capturing a graph
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    const bool capturing = cudaStreamIsCapturing((cudaStream_t)stream, &cap) != cudaSuccess || cap != cudaStreamCaptureStatusNone;
    const long long chain_expect = (c->chain_ok && !capturing && c->pdl_opt != 0) ? (long long)c->step_done : -1;
    c->view.l2_keep = l2_keep_fraction(c, seq_ids, n_seqs);
    MM_CUDA(c, launch_step_mma(c->view, list, k_new, v_new, q, out, lse, sm_scale, layer_begin, layer_end, !opens, grid,
                               c->pdl_opt != 0, chain_expect, (cudaStream_t)stream, &li));
    note(c, li);
    if (!capturing) {
      c->step_done += (uint32_t)li.grid;
      c->chain_ok = true;
    }
    if (opens) {
      const int32_t p = c->desc.page_size;
      for (int i = 0; i < n_seqs; ++i) {  // host mirror of the append (validated by check_step) ...
        HostSeq& hs = c->seqs[seq_ids[i]];
        c->free_pages -= blocks_for(hs.sp.len + 1, p) - blocks_for(hs.sp.len, p);
        hs.sp.len += 1;
      }
      mirror_evict(c, seq_ids, n_seqs);  // ... and of the eviction
      c->stats.append_calls += 1;
    }
    for (int i = 0; i < n_seqs; ++i) open_step_mark(c, c->seqs[seq_ids[i]], layer_begin, layer_end, opens);
    c->stats.attn_calls += 1;
    c->stats.attn_grid = li.grid;
    c->stats.attn_smem_bytes = li.smem;
    c->stats.attn_variant = variant;
    return MURMUR_OK;
  }
  const bool fuse = opens && c->fuse_step_opt != 0;  // n_seqs <= 128 (check_step): one append launch
  st = append_impl(c, seq_ids, ones, n_seqs, k_new, v_new, layer_begin, layer_end, fuse, stream);
  if (st != MURMUR_OK) return st;
  if (opens && !fuse) {
    st = murmur_kv_evict(c, seq_ids, n_seqs, stream);
    if (st != MURMUR_OK) return st;
  }
  for (int i = 0; i < n_seqs; ++i) open_step_mark(c, c->seqs[seq_ids[i]], layer_begin, layer_end, opens);
  return murmur_decode_attn(c, seq_ids, n_seqs, q, out, lse, layer_begin, layer_end, sm_scale, stream);
}

murmur_status_t murmur_decode_step(murmur_cache_t* c, const int32_t* seq_ids, int32_t n_seqs, const void* k_new,
                                   const void* v_new, const void* q, void* out, float* lse, float sm_scale,
                                   void* stream) {
  if (!c) return MURMUR_ERR_INVALID_ARG;
  return step_layers_impl(c, seq_ids, n_seqs, k_new, v_new, q, out, lse, 0, c->desc.n_layers, sm_scale, stream);
}

murmur_status_t murmur_decode_step_layers(murmur_cache_t* c, const int32_t* seq_ids, int32_t n_seqs, const void* k_new,
                                          const void* v_new, const void* q, void* out, float* lse, int32_t layer_begin,
                                          int32_t layer_end, float sm_scale, void* stream) {
  return step_layers_impl(c, seq_ids, n_seqs, k_new, v_new, q, out, lse, layer_begin, layer_end, sm_scale, stream);
}

murmur_status_t murmur_decode_step_chunked(murmur_cache_t* c, const int32_t* seq_ids, int32_t n_seqs, const void* k_new,
                                           const void* v_new, const void* q, void* out, float* lse,
                                           int32_t layers_per_launch, float sm_scale, void* stream) {
  if (!c || layers_per_launch < 1) return MURMUR_ERR_INVALID_ARG;
  if (n_seqs < 1 || !k_new || !v_new || !q || !out) return MURMUR_ERR_INVALID_ARG;
  const int L = c->desc.n_layers;
  const size_t kv_l = (size_t)n_seqs * c->desc.n_kv_heads * kRowBytes;  // bytes of one layer of k_new / v_new
  const size_t q_l = (size_t)n_seqs * c->desc.n_q_heads * kRowBytes;    // ... of q / out
  const size_t lse_l = (size_t)n_seqs * c->desc.n_q_heads;              // floats
  for (int lb = 0; lb < L; lb += layers_per_launch) {
    const int le = lb + layers_per_launch < L ? lb + layers_per_launch : L;
    // the opening range validates the whole step (all-or-nothing) before anything is enqueued
    murmur_status_t st = step_layers_impl(c, seq_ids, n_seqs, (const uint8_t*)k_new + lb * kv_l,
                                          (const uint8_t*)v_new + lb * kv_l, (const uint8_t*)q + lb * q_l,
                                          (uint8_t*)out + lb * q_l, lse ? lse + lb * lse_l : nullptr, lb, le, sm_scale,
                                          stream);
    if (st != MURMUR_OK) return st;
  }
  return MURMUR_OK;
}

murmur_status_t murmur_decode_step_host(murmur_cache_t* c, const int32_t* seq_ids, int32_t n_seqs,
                                        const void* k_new_host, const void* v_new_host, const void* q_host,
                                        void* out_host, float sm_scale, void* stream) {
  if (!c || !k_new_host || !v_new_host || !q_host || !out_host) return MURMUR_ERR_INVALID_ARG;
  MM_GUARD(c, stream);
  if (!(sm_scale > 0.f)) return MURMUR_ERR_INVALID_ARG;
  if (n_seqs < 1 || n_seqs > c->cv.stage_seqs) return MURMUR_ERR_INVALID_ARG;
  // validate before any copy so that a failing call leaves everything untouched
  murmur_status_t st = check_step(c, seq_ids, n_seqs);
  if (st != MURMUR_OK) return st;
  cudaStream_t s = (cudaStream_t)stream;
  const size_t kv_b = (size_t)c->desc.n_layers * n_seqs * c->desc.n_kv_heads * kRowBytes;
  const size_t q_b = (size_t)c->desc.n_layers * n_seqs * c->desc.n_q_heads * kRowBytes;
  // Zero-copy path: when all four buffers are page-locked (cudaHostAlloc / cudaHostRegister / torch pin_memory)
  // the step kernel works on their device-mapped addresses directly - Q and the new K/V rows arrive by the same
  // bulk copies straight from host memory while the pool streams from HBM, and `out` is stored to the host
  // buffer by the kernel.  The bytes still cross PCIe inside the call; no staging copy on either side.
  if (c->host_zero_copy_opt) {
    const void* hp[4] = {k_new_host, v_new_host, q_host, out_host};
    void* dp[4] = {nullptr, nullptr, nullptr, nullptr};
    bool mapped = true;
    for (int i = 0; i < 4 && mapped; ++i) {
      cudaPointerAttributes at{};
      if (cudaPointerGetAttributes(&at, hp[i]) != cudaSuccess) {
        (void)cudaGetLastError();  // unregistered host memory on older drivers: not an error here
        mapped = false;
      } else if (at.type != cudaMemoryTypeHost || at.devicePointer == nullptr || ((uintptr_t)at.devicePointer & 15)) {
        mapped = false;
      } else {
        dp[i] = at.devicePointer;
      }
    }
    if (mapped) {
      c->stats.host_zero_copy_steps += 1;
      return murmur_decode_step(c, seq_ids, n_seqs, dp[0], dp[1], dp[2], dp[3], nullptr, sm_scale, stream);
    }
  }
  uint8_t* dk = c->ws + c->cv.stage_k;
  uint8_t* dv = c->ws + c->cv.stage_v;
  uint8_t* dq = c->ws + c->cv.stage_q;
  uint8_t* dout = c->ws + c->cv.stage_out;
  const uint8_t* hk = reinterpret_cast<const uint8_t*>(k_new_host);
  const uint8_t* hv = reinterpret_cast<const uint8_t*>(v_new_host);
  const uint8_t* hq = reinterpret_cast<const uint8_t*>(q_host);
  if (hv == hk + kv_b && hq == hv + kv_b && dv == dk + kv_b && dq == dv + kv_b) {
    // k, v, q packed back to back on the host (and in the staging area): one copy instead of three
    MM_CUDA(c, cudaMemcpyAsync(dk, hk, 2 * kv_b + q_b, cudaMemcpyHostToDevice, s));
  } else {
    MM_CUDA(c, cudaMemcpyAsync(dk, hk, kv_b, cudaMemcpyHostToDevice, s));
    MM_CUDA(c, cudaMemcpyAsync(dv, hv, kv_b, cudaMemcpyHostToDevice, s));
    MM_CUDA(c, cudaMemcpyAsync(dq, hq, q_b, cudaMemcpyHostToDevice, s));
  }
  st = murmur_decode_step(c, seq_ids, n_seqs, dk, dv, dq, dout, nullptr, sm_scale, stream);
  if (st != MURMUR_OK) return st;
  MM_CUDA(c, cudaMemcpyAsync(out_host, dout, q_b, cudaMemcpyDeviceToHost, s));
  return MURMUR_OK;
}

// ---- prefill ------------------------------------------------------------------------------------
murmur_status_t murmur_prefill_attn(murmur_cache_t* c, int32_t seq, int32_t pos_begin, int32_t pos_end, const void* q,
                                    void* out, float* lse, int32_t layer_begin, int32_t layer_end, float sm_scale,
                                    void* stream) {
  murmur_status_t st = check_seq(c, seq);
  if (st != MURMUR_OK) return st;
  MM_GUARD(c, stream);
  if (!q || !out) return MURMUR_ERR_INVALID_ARG;
  if (layer_begin < 0 || layer_end > c->desc.n_layers || layer_begin >= layer_end) return MURMUR_ERR_INVALID_ARG;
  if (!(sm_scale > 0.f)) return MURMUR_ERR_INVALID_ARG;
  if (c->desc.page_size < 16) return MURMUR_ERR_UNSUPPORTED;
  const HostSeq& hs = c->seqs[seq];
  if (hs.indexed) return MURMUR_ERR_STATE;
  if (pos_begin < 0 || pos_begin >= pos_end || pos_end > hs.sp.len) return MURMUR_ERR_INVALID_ARG;
  if (hs.freed_blocks != 0) return MURMUR_ERR_STATE;  // something below pos_end may be gone
  LaunchInfo li{};
  if (c->prefill_variant_opt == MURMUR_PREFILL_MMA_SYNC) {
    MM_CUDA(c, launch_prefill_attn(c->view, seq, pos_begin, pos_end - pos_begin, q, out, lse, layer_begin, layer_end,
                                   sm_scale, (cudaStream_t)stream, &li));
  } else {  // tcgen05 + tensor memory (the tensor maps need 16-byte aligned bases)
    if (((uintptr_t)q | (uintptr_t)out) & 15) return MURMUR_ERR_INVALID_ARG;
    MM_CUDA(c, launch_prefill_attn_umma(c->view, seq, pos_begin, pos_end - pos_begin, q, out, lse, layer_begin,
                                        layer_end, sm_scale, c->sm_count, (cudaStream_t)stream, &li));
  }
  note(c, li);
  return MURMUR_OK;
}

// ---- analysis -----------------------------------------------------------------------------------
static long long profile_stride(murmur_cache_t* c, const int32_t* seq_ids, int32_t n_seqs) {
  int32_t mx = 1;
  for (int i = 0; i < n_seqs; ++i) mx = c->seqs[seq_ids[i]].sp.len > mx ? c->seqs[seq_ids[i]].sp.len : mx;
  return ((long long)mx + 31) / 32 * 32;
}

size_t murmur_profile_scratch_bytes(murmur_cache_t* c, const int32_t* seq_ids, int32_t n_seqs, int32_t layer_begin,
                                    int32_t layer_end) {
  if (!c || n_seqs < 1 || n_seqs > kMaxSeqsPerLaunch) return 0;
  if (check_ids(c, seq_ids, n_seqs) != MURMUR_OK) return 0;
  if (layer_begin < 0 || layer_end > c->desc.n_layers || layer_begin >= layer_end) return 0;
  return (size_t)(layer_end - layer_begin) * n_seqs * c->desc.n_q_heads * (size_t)profile_stride(c, seq_ids, n_seqs) * 4;
}

murmur_status_t murmur_attn_profile(murmur_cache_t* c, const int32_t* seq_ids, int32_t n_seqs, const void* q,
                                    const murmur_policy_t* cand, float mass_frac, void* out, void* scratch,
                                    size_t scratch_bytes, int32_t layer_begin, int32_t layer_end, float sm_scale,
                                    void* stream) {
  if (!c || !q || !out || !scratch) return MURMUR_ERR_INVALID_ARG;
  if (n_seqs < 1 || n_seqs > kMaxSeqsPerLaunch) return MURMUR_ERR_INVALID_ARG;
  murmur_status_t st = check_ids(c, seq_ids, n_seqs);
  if (st != MURMUR_OK) return st;
  if (layer_begin < 0 || layer_end > c->desc.n_layers || layer_begin >= layer_end) return MURMUR_ERR_INVALID_ARG;
  if (!(sm_scale > 0.f) || !(mass_frac > 0.f) || mass_frac > 1.f) return MURMUR_ERR_INVALID_ARG;
  if (cand && (cand->w_speech < 0 || cand->delay < 0 || cand->n_sink_speech < 0 || cand->w_out < 0 || cand->n_sink_out < 0))
    return MURMUR_ERR_INVALID_ARG;
  for (int i = 0; i < n_seqs; ++i)
    if (c->seqs[seq_ids[i]].sp.len < 1) return MURMUR_ERR_STATE;
  if (scratch_bytes < murmur_profile_scratch_bytes(c, seq_ids, n_seqs, layer_begin, layer_end)) return MURMUR_ERR_INVALID_ARG;
  SeqList list;
  list.n = n_seqs;
  for (int i = 0; i < n_seqs; ++i) list.ids[i] = seq_ids[i];
  SeqParams cs{};
  if (cand) {
    cs.w_s = cand->w_speech; cs.d = cand->delay; cs.k_s = cand->n_sink_speech; cs.w_o = cand->w_out; cs.k_o = cand->n_sink_out;
  }
  LaunchInfo li{};
  MM_CUDA(c, launch_attn_profile(c->view, list, 0, n_seqs, q, cand ? &cs : nullptr, mass_frac, out,
                                 reinterpret_cast<float*>(scratch), profile_stride(c, seq_ids, n_seqs), layer_begin,
                                 layer_end, sm_scale, nullptr, (cudaStream_t)stream, &li));
  note(c, li);
  return MURMUR_OK;
}

// The profile with the library's built-in scratch (attn_profile.cu): for callers that cannot allocate - see murmur.h.
// Validation is that of murmur_attn_profile; the scratch need is checked against the fixed array before any launch.
murmur_status_t murmur_attn_profile_noalloc(murmur_cache_t* c, const int32_t* seq_ids, int32_t n_seqs, const void* q,
                                            const murmur_policy_t* cand, float mass_frac, void* out,
                                            int32_t layer_begin, int32_t layer_end, float sm_scale, void* stream) {
  if (!c || !q || !out) return MURMUR_ERR_INVALID_ARG;
  if (n_seqs < 1 || n_seqs > kMaxSeqsPerLaunch) return MURMUR_ERR_INVALID_ARG;
  murmur_status_t st = check_ids(c, seq_ids, n_seqs);
  if (st != MURMUR_OK) return st;
  if (layer_begin < 0 || layer_end > c->desc.n_layers || layer_begin >= layer_end) return MURMUR_ERR_INVALID_ARG;
  if (!(sm_scale > 0.f) || !(mass_frac > 0.f) || mass_frac > 1.f) return MURMUR_ERR_INVALID_ARG;
  if (cand && (cand->w_speech < 0 || cand->delay < 0 || cand->n_sink_speech < 0 || cand->w_out < 0 || cand->n_sink_out < 0))
    return MURMUR_ERR_INVALID_ARG;
  for (int i = 0; i < n_seqs; ++i)
    if (c->seqs[seq_ids[i]].sp.len < 1) return MURMUR_ERR_STATE;
  const size_t need = murmur_profile_scratch_bytes(c, seq_ids, n_seqs, layer_begin, layer_end);
  if (need == 0) return MURMUR_ERR_INVALID_ARG;
  if (need > (size_t)MURMUR_PROFILE_NOALLOC_MAX_BYTES) return MURMUR_ERR_SCRATCH_LIMIT;
  SeqList list;
  list.n = n_seqs;
  for (int i = 0; i < n_seqs; ++i) list.ids[i] = seq_ids[i];
  SeqParams cs{};
  if (cand) {
    cs.w_s = cand->w_speech; cs.d = cand->delay; cs.k_s = cand->n_sink_speech; cs.w_o = cand->w_out; cs.k_o = cand->n_sink_out;
  }
  LaunchInfo li{};
  MM_CUDA(c, launch_attn_profile_noalloc(c->view, list, n_seqs, q, cand ? &cs : nullptr, mass_frac, out,
                                         profile_stride(c, seq_ids, n_seqs), need, layer_begin, layer_end, sm_scale,
                                         (cudaStream_t)stream, &li));
  note(c, li);
  return MURMUR_OK;
}

// ---- general index-set eviction (indexed mode) ------------------------------------------------------
static size_t idx_len_bytes(const murmur_cache_desc_t* d) {
  return align_up((size_t)d->max_seqs * d->n_layers * d->n_kv_heads * 4);
}

size_t murmur_indexed_bytes(const murmur_cache_desc_t* d) {
  if (!geometry_ok(d)) return 0;
  const size_t cap = (size_t)d->max_blocks_per_seq * d->page_size;
  return kAlign + idx_len_bytes(d) + align_up((size_t)d->max_seqs * d->n_layers * d->n_kv_heads * cap * 4);
}

murmur_status_t murmur_indexed_enable(murmur_cache_t* c, void* buffer, size_t bytes, void* stream) {
  if (!c || !buffer) return MURMUR_ERR_INVALID_ARG;
  if (((uintptr_t)buffer & (kAlign - 1)) || bytes < murmur_indexed_bytes(&c->desc)) return MURMUR_ERR_INVALID_ARG;
  for (const HostSeq& hs : c->seqs)
    if (hs.indexed) return MURMUR_ERR_STATE;  // tables in use
  uint8_t* b = reinterpret_cast<uint8_t*>(buffer);
  MM_CUDA(c, cudaMemsetAsync(b, 0, kAlign + idx_len_bytes(&c->desc), (cudaStream_t)stream));
  c->idx_moved = reinterpret_cast<unsigned long long*>(b);
  c->idx.len = reinterpret_cast<int32_t*>(b + kAlign);
  c->idx.pos = reinterpret_cast<int32_t*>(b + kAlign + idx_len_bytes(&c->desc));
  c->idx.cap = c->desc.max_blocks_per_seq * c->desc.page_size;
  return MURMUR_OK;
}

size_t murmur_select_scratch_bytes(murmur_cache_t* c, int32_t seq) {
  if (check_seq(c, seq) != MURMUR_OK || c->seqs[seq].indexed) return 0;
  const size_t stride = (size_t)profile_stride(c, &seq, 1);
  return (size_t)c->desc.n_layers * c->desc.n_q_heads * stride * 4 + align_up((size_t)c->desc.n_layers * c->desc.n_kv_heads * stride);
}

murmur_status_t murmur_select_mass_sets(murmur_cache_t* c, int32_t seq, const void* q, float mass_frac, int32_t n_recent,
                                        int32_t* sel_pos, int32_t* sel_cnt, int32_t cap, void* scratch, size_t scratch_bytes,
                                        float sm_scale, void* stream) {
  murmur_status_t st = check_seq(c, seq);
  if (st != MURMUR_OK) return st;
  if (!q || !sel_pos || !sel_cnt || !scratch || cap < 1 || n_recent < 0) return MURMUR_ERR_INVALID_ARG;
  if (!(sm_scale > 0.f) || !(mass_frac > 0.f) || mass_frac > 1.f) return MURMUR_ERR_INVALID_ARG;
  const HostSeq& hs = c->seqs[seq];
  if (hs.indexed || hs.sp.len < 1) return MURMUR_ERR_STATE;  // sets are selected over a positional cache
  if (scratch_bytes < murmur_select_scratch_bytes(c, seq)) return MURMUR_ERR_INVALID_ARG;
  const long long stride = profile_stride(c, &seq, 1);
  float* sc = reinterpret_cast<float*>(scratch);
  uint8_t* mask = reinterpret_cast<uint8_t*>(scratch) + (size_t)c->desc.n_layers * c->desc.n_q_heads * (size_t)stride * 4;
  SeqList list;
  list.n = 1;
  list.ids[0] = seq;
  LaunchInfo li{};
  MM_CUDA(c, launch_attn_profile(c->view, list, 0, 1, q, nullptr, mass_frac, nullptr, sc, stride, 0, c->desc.n_layers,
                                 sm_scale, mask, (cudaStream_t)stream, &li));
  MM_CUDA(c, launch_select_compact(c->view, seq, mask, stride, n_recent, sel_pos, sel_cnt, cap, (cudaStream_t)stream, &li));
  note(c, li);
  return MURMUR_OK;
}

murmur_status_t murmur_kv_evict_indexed(murmur_cache_t* c, int32_t seq, const int32_t* sel_pos, const int32_t* sel_cnt,
                                        int32_t cap, int64_t* bytes_moved_out, void* stream) {
  murmur_status_t st = check_seq(c, seq);
  if (st != MURMUR_OK) return st;
  MM_GUARD(c, stream);
  if (!sel_pos || !sel_cnt || cap < 1) return MURMUR_ERR_INVALID_ARG;
  if (!c->idx.pos) return MURMUR_ERR_STATE;  // murmur_indexed_enable first
  HostSeq& hs = c->seqs[seq];
  if (!hs.indexed && (hs.sp.len < 1 || hs.evict_len != hs.sp.len)) return MURMUR_ERR_STATE;  // live page list must be current
  cudaStream_t s = (cudaStream_t)stream;
  const int n_slabs = c->desc.n_layers * c->desc.n_kv_heads;
  std::vector<int32_t> cnt(n_slabs);
  // The sets are checked on the device BEFORE anything moves (sizes, strict ascending order, every position held by
  // its slab): the compaction is in place, so a bad set found half-way could not be undone.  The verdict word shares
  // the 256-byte block of the moved-rows counter and is read in the synchronisation that fetches the set sizes.
  int* bad_dev = reinterpret_cast<int*>(c->idx_moved) + 4;
  int32_t bad = 0;
  LaunchInfo lv{};
  MM_CUDA(c, cudaMemsetAsync(bad_dev, 0, 4, s));
  MM_CUDA(c, launch_indexed_validate(c->view, c->idx, seq, sel_pos, sel_cnt, cap, !hs.indexed, bad_dev, s, &lv));
  note(c, lv);
  MM_CUDA(c, cudaMemcpyAsync(cnt.data(), sel_cnt, (size_t)n_slabs * 4, cudaMemcpyDeviceToHost, s));
  MM_CUDA(c, cudaMemcpyAsync(&bad, bad_dev, 4, cudaMemcpyDeviceToHost, s));
  MM_CUDA(c, cudaStreamSynchronize(s));
  const int32_t held = hs.indexed ? hs.idx_max_len : hs.sp.len;  // a slab cannot grow by eviction
  int32_t mx = 0;
  for (int i = 0; i < n_slabs; ++i) {
    if (cnt[i] < 1 || cnt[i] > cap || cnt[i] > held) return MURMUR_ERR_INVALID_ARG;
    mx = cnt[i] > mx ? cnt[i] : mx;
  }
  if (bad != 0) return MURMUR_ERR_INVALID_ARG;  // nothing moved, no page freed, the sequence keeps its mode
  const int32_t p = c->desc.page_size;
  const int32_t blocks_held = hs.indexed ? hs.idx_blocks : blocks_for(hs.sp.len, p) - hs.freed_blocks;
  const int32_t nb_new = blocks_for(mx, p);
  if (nb_new > blocks_held) return MURMUR_ERR_INVALID_ARG;
  MM_CUDA(c, cudaMemsetAsync(c->idx_moved, 0, 8, s));
  LaunchInfo li{};
  MM_CUDA(c, launch_indexed_defrag(c->view, c->idx, seq, sel_pos, sel_cnt, cap, !hs.indexed, c->idx_moved, s, &li));
  note(c, li);
  unsigned long long moved = 0;
  MM_CUDA(c, cudaMemcpyAsync(&moved, c->idx_moved, 8, cudaMemcpyDeviceToHost, s));
  MM_CUDA(c, cudaStreamSynchronize(s));
  if (bytes_moved_out) *bytes_moved_out = (int64_t)moved * 2 * kRowBytes;
  c->free_pages += blocks_held - nb_new;
  c->stats.free_pages = c->free_pages;
  hs.indexed = true;
  hs.idx_blocks = nb_new;
  hs.idx_max_len = mx;
  return MURMUR_OK;
}

murmur_status_t murmur_kv_append_indexed(murmur_cache_t* c, const int32_t* seq_ids, int32_t n_seqs, const void* k_new,
                                         const void* v_new, void* stream) {
  if (!c || !k_new || !v_new) return MURMUR_ERR_INVALID_ARG;
  MM_GUARD(c, stream);
  if (n_seqs < 1 || n_seqs > kMaxSeqsPerLaunch) return MURMUR_ERR_INVALID_ARG;
  murmur_status_t st = check_ids(c, seq_ids, n_seqs, 1);
  if (st != MURMUR_OK) return st;
  const int32_t p = c->desc.page_size;
  int64_t need = 0;
  for (int i = 0; i < n_seqs; ++i) {
    const HostSeq& hs = c->seqs[seq_ids[i]];
    if (hs.idx_max_len + 1 > c->idx.cap) return MURMUR_ERR_STATE;
    need += blocks_for(hs.idx_max_len + 1, p) - hs.idx_blocks;
  }
  if (need > c->free_pages) return MURMUR_ERR_OOM_PAGES;  // all-or-nothing
  SeqList list;
  list.n = n_seqs;
  for (int i = 0; i < n_seqs; ++i) list.ids[i] = seq_ids[i];
  LaunchInfo li{};
  MM_CUDA(c, launch_indexed_append(c->view, c->idx, list, k_new, v_new, (cudaStream_t)stream, &li));
  note(c, li);
  for (int i = 0; i < n_seqs; ++i) {
    HostSeq& hs = c->seqs[seq_ids[i]];
    hs.idx_blocks = blocks_for(hs.idx_max_len + 1, p);
    hs.idx_max_len += 1;
  }
  c->free_pages -= need;
  c->stats.free_pages = c->free_pages;
  c->stats.append_calls += 1;
  return MURMUR_OK;
}

murmur_status_t murmur_decode_attn_indexed(murmur_cache_t* c, const int32_t* seq_ids, int32_t n_seqs, const void* q,
                                           void* out, float* lse, float sm_scale, void* stream) {
  if (!c || !q || !out) return MURMUR_ERR_INVALID_ARG;
  MM_GUARD(c, stream);
  if (n_seqs < 1 || n_seqs > kMaxSeqsPerLaunch || !(sm_scale > 0.f)) return MURMUR_ERR_INVALID_ARG;
  murmur_status_t st = check_ids(c, seq_ids, n_seqs, 1);
  if (st != MURMUR_OK) return st;
  SeqList list;
  list.n = n_seqs;
  for (int i = 0; i < n_seqs; ++i) list.ids[i] = seq_ids[i];
  LaunchInfo li{};
  // tensor cores whenever a page holds whole 16-row MMA slices (same rule and option as the positional call)
  int variant = c->attn_variant_opt;
  if (variant == MURMUR_ATTN_AUTO) variant = (c->desc.page_size >= 16) ? MURMUR_ATTN_MMA : MURMUR_ATTN_GENERIC;
  if (variant == MURMUR_ATTN_MMA && c->desc.page_size < 16) return MURMUR_ERR_UNSUPPORTED;
  if (variant == MURMUR_ATTN_MMA) {
    MM_CUDA(c, launch_indexed_attn_mma(c->view, c->idx, list, q, out, lse, sm_scale, (cudaStream_t)stream, &li));
  } else {
    MM_CUDA(c, launch_indexed_attn(c->view, c->idx, list, q, out, lse, sm_scale, (cudaStream_t)stream, &li));
  }
  note(c, li);
  c->stats.attn_calls += 1;
  return MURMUR_OK;
}

murmur_status_t murmur_kv_get_indexed(murmur_cache_t* c, int32_t seq, int32_t layer, int32_t kv_head, int32_t* pos_out,
                                      int32_t cap, int32_t* n_out, void* stream) {
  murmur_status_t st = check_seq(c, seq);
  if (st != MURMUR_OK) return st;
  if (!c->seqs[seq].indexed) return MURMUR_ERR_STATE;
  if (!n_out || cap < 0 || (cap > 0 && !pos_out)) return MURMUR_ERR_INVALID_ARG;
  if (layer < 0 || layer >= c->desc.n_layers || kv_head < 0 || kv_head >= c->desc.n_kv_heads) return MURMUR_ERR_INVALID_ARG;
  MM_CUDA(c, cudaStreamSynchronize((cudaStream_t)stream));
  const size_t slab = (size_t)seq * c->desc.n_layers * c->desc.n_kv_heads + (size_t)layer * c->desc.n_kv_heads + kv_head;
  int32_t n = 0;
  MM_CUDA(c, cudaMemcpy(&n, c->idx.len + slab, 4, cudaMemcpyDeviceToHost));
  *n_out = n;
  if (n > cap) return MURMUR_ERR_INVALID_ARG;
  if (n > 0) MM_CUDA(c, cudaMemcpy(pos_out, c->idx.pos + slab * c->idx.cap, (size_t)n * 4, cudaMemcpyDeviceToHost));
  return MURMUR_OK;
}

murmur_status_t murmur_kv_gather_indexed(murmur_cache_t* c, int32_t seq, void* k_out, void* v_out, int32_t cap_rows,
                                         void* stream) {
  murmur_status_t st = check_seq(c, seq);
  if (st != MURMUR_OK) return st;
  if (!c->seqs[seq].indexed) return MURMUR_ERR_STATE;
  if (!k_out || !v_out || cap_rows < 1) return MURMUR_ERR_INVALID_ARG;
  LaunchInfo li{};
  MM_CUDA(c, launch_indexed_gather(c->view, c->idx, seq, k_out, v_out, cap_rows, (cudaStream_t)stream, &li));
  note(c, li);
  MM_CUDA(c, cudaStreamSynchronize((cudaStream_t)stream));
  return MURMUR_OK;
}

// ---- introspection ------------------------------------------------------------------------------
static murmur_status_t check_seq(murmur_cache_t* c, int32_t seq) {
  if (!c) return MURMUR_ERR_INVALID_ARG;
  if (seq < 0 || seq >= c->desc.max_seqs) return MURMUR_ERR_INVALID_ARG;
  if (!c->seqs[seq].active) return MURMUR_ERR_STATE;
  return MURMUR_OK;
}

static murmur_status_t read_seqdev(murmur_cache_t* c, int32_t seq, SeqDev* sd, cudaStream_t s) {
  MM_CUDA(c, cudaStreamSynchronize(s));
  MM_CUDA(c, cudaMemcpy(sd, c->view.seqs + seq, sizeof(SeqDev), cudaMemcpyDeviceToHost));
  return MURMUR_OK;
}

murmur_status_t murmur_seq_get_state(murmur_cache_t* c, int32_t seq, int32_t* state_out, void* stream) {
  murmur_status_t st = check_seq(c, seq);
  if (st != MURMUR_OK) return st;
  if (!state_out) return MURMUR_ERR_INVALID_ARG;
  SeqDev sd;
  st = read_seqdev(c, seq, &sd, (cudaStream_t)stream);
  if (st != MURMUR_OK) return st;
  state_out[0] = sd.len;
  state_out[1] = sd.len - (sd.P + sd.S + sd.M) > 0 ? sd.len - (sd.P + sd.S + sd.M) : 0;
  state_out[2] = sd.n_live;
  state_out[3] = sd.n_runs;
  state_out[4] = sd.n_tiles;
  state_out[5] = sd.n_retained;
  return MURMUR_OK;
}

murmur_status_t murmur_kv_get_retained(murmur_cache_t* c, int32_t seq, int32_t* pos_out, int32_t cap, int32_t* n_out,
                                       void* stream) {
  murmur_status_t st = check_seq(c, seq);
  if (st != MURMUR_OK) return st;
  if (!n_out || cap < 0 || (cap > 0 && !pos_out)) return MURMUR_ERR_INVALID_ARG;
  SeqDev sd;
  st = read_seqdev(c, seq, &sd, (cudaStream_t)stream);
  if (st != MURMUR_OK) return st;
  *n_out = sd.n_retained;
  if (sd.n_retained > cap) return MURMUR_ERR_INVALID_ARG;
  if (sd.n_retained == 0) return MURMUR_OK;
  if ((size_t)sd.n_retained > c->cv.scratch_ints) return MURMUR_ERR_STATE;
  int32_t* scratch = reinterpret_cast<int32_t*>(c->ws + c->cv.scratch);
  LaunchInfo li{};
  MM_CUDA(c, launch_expand_retained(c->view, seq, scratch, (int)c->cv.scratch_ints, (cudaStream_t)stream, &li));
  note(c, li);
  MM_CUDA(c, cudaStreamSynchronize((cudaStream_t)stream));
  MM_CUDA(c, cudaMemcpy(pos_out, scratch, (size_t)sd.n_retained * 4, cudaMemcpyDeviceToHost));
  return MURMUR_OK;
}

murmur_status_t murmur_kv_get_page_list(murmur_cache_t* c, int32_t seq, int32_t* pages_out, int32_t* blocks_out,
                                        int32_t cap, int32_t* n_out, void* stream) {
  murmur_status_t st = check_seq(c, seq);
  if (st != MURMUR_OK) return st;
  if (!n_out || cap < 0) return MURMUR_ERR_INVALID_ARG;
  SeqDev sd;
  st = read_seqdev(c, seq, &sd, (cudaStream_t)stream);
  if (st != MURMUR_OK) return st;
  *n_out = sd.n_live;
  if (sd.n_live > cap) return MURMUR_ERR_INVALID_ARG;
  const size_t off = (size_t)seq * c->desc.max_blocks_per_seq;
  if (pages_out && sd.n_live)
    MM_CUDA(c, cudaMemcpy(pages_out, c->view.live_pages + off, (size_t)sd.n_live * 4, cudaMemcpyDeviceToHost));
  if (blocks_out && sd.n_live)
    MM_CUDA(c, cudaMemcpy(blocks_out, c->view.live_blocks + off, (size_t)sd.n_live * 4, cudaMemcpyDeviceToHost));
  return MURMUR_OK;
}

murmur_status_t murmur_kv_get_runs(murmur_cache_t* c, int32_t seq, int32_t* runs_out, int32_t cap_runs, int32_t* n_out,
                                   void* stream) {
  murmur_status_t st = check_seq(c, seq);
  if (st != MURMUR_OK) return st;
  if (!n_out || !runs_out) return MURMUR_ERR_INVALID_ARG;
  SeqDev sd;
  st = read_seqdev(c, seq, &sd, (cudaStream_t)stream);
  if (st != MURMUR_OK) return st;
  *n_out = sd.n_runs;
  if (sd.n_runs > cap_runs) return MURMUR_ERR_INVALID_ARG;
  for (int r = 0; r < sd.n_runs; ++r)
    for (int k = 0; k < 3; ++k) runs_out[3 * r + k] = sd.runs[r][k];
  return MURMUR_OK;
}

murmur_status_t murmur_kv_get_free_stack(murmur_cache_t* c, int32_t* pages_out, int64_t cap, int64_t* n_out,
                                         void* stream) {
  if (!c || !n_out) return MURMUR_ERR_INVALID_ARG;
  MM_CUDA(c, cudaStreamSynchronize((cudaStream_t)stream));
  int32_t top = 0;
  MM_CUDA(c, cudaMemcpy(&top, c->view.ctrl + kCtrlFreeTop, 4, cudaMemcpyDeviceToHost));
  *n_out = top;
  if (top > cap) return MURMUR_ERR_INVALID_ARG;
  if (pages_out && top > 0)
    MM_CUDA(c, cudaMemcpy(pages_out, c->view.free_stack, (size_t)top * 4, cudaMemcpyDeviceToHost));
  return MURMUR_OK;
}

murmur_status_t murmur_kv_gather(murmur_cache_t* c, int32_t seq, const int32_t* positions, int32_t n,
                                 int32_t layer_begin, int32_t layer_end, void* k_out, void* v_out, void* stream) {
  murmur_status_t st = check_seq(c, seq);
  if (st != MURMUR_OK) return st;
  if (c->seqs[seq].indexed) return MURMUR_ERR_STATE;  // rows are addressed by slot there: murmur_kv_gather_indexed
  if (!positions || n < 0 || !k_out || !v_out) return MURMUR_ERR_INVALID_ARG;
  if (layer_begin < 0 || layer_end > c->desc.n_layers || layer_begin >= layer_end) return MURMUR_ERR_INVALID_ARG;
  if ((size_t)n > c->cv.scratch_ints) return MURMUR_ERR_INVALID_ARG;
  for (int i = 0; i < n; ++i)
    if (positions[i] < 0 || positions[i] >= c->seqs[seq].sp.len) return MURMUR_ERR_INVALID_ARG;
  if (n == 0) return MURMUR_OK;
  int32_t* scratch = reinterpret_cast<int32_t*>(c->ws + c->cv.scratch);
  cudaStream_t s = (cudaStream_t)stream;
  MM_CUDA(c, cudaStreamSynchronize(s));
  MM_CUDA(c, cudaMemcpy(scratch, positions, (size_t)n * 4, cudaMemcpyHostToDevice));
  LaunchInfo li{};
  MM_CUDA(c, launch_gather(c->view, seq, scratch, n, layer_begin, layer_end, k_out, v_out, s, &li));
  note(c, li);
  MM_CUDA(c, cudaStreamSynchronize(s));
  return MURMUR_OK;
}

// Re-reads the integer state the host mirror shadows (lengths, free-stack height) from the device.
murmur_status_t murmur_mirror_sync(murmur_cache_t* c, void* stream) {
  if (!c) return MURMUR_ERR_INVALID_ARG;
  cudaStream_t s = (cudaStream_t)stream;
  MM_CUDA(c, cudaStreamSynchronize(s));
  std::vector<SeqDev> dev(c->desc.max_seqs);
  MM_CUDA(c, cudaMemcpy(dev.data(), c->view.seqs, dev.size() * sizeof(SeqDev), cudaMemcpyDeviceToHost));
  int32_t top = 0;
  MM_CUDA(c, cudaMemcpy(&top, c->view.ctrl + kCtrlFreeTop, 4, cudaMemcpyDeviceToHost));
  for (int i = 0; i < c->desc.max_seqs; ++i) {
    HostSeq& hs = c->seqs[i];
    const SeqDev& sd = dev[i];
    if (!hs.active || !sd.active) continue;  // sequences begin and end through the API only
    if (hs.indexed) {
      hs.idx_blocks = sd.idx_blocks;
      hs.idx_max_len = sd.idx_max_len;
      continue;
    }
    if (sd.len != hs.sp.len) {  // steps ran on the device that the mirror has not seen: every step ends with its eviction
      hs.sp.len = sd.len;
      hs.evict_len = sd.len;
      hs.freed_blocks = dead_block_count(hs.sp, c->desc.page_size);
    }
  }
  c->free_pages = top;
  c->stats.free_pages = c->free_pages;
  int32_t done = 0;  // replayed step launches counted on the device only
  MM_CUDA(c, cudaMemcpy(&done, c->view.ctrl + kCtrlStepDone, 4, cudaMemcpyDeviceToHost));
  c->step_done = (uint32_t)done;
  c->chain_ok = false;
  for (HostSeq& hs : c->seqs) hs.open_len = -1;  // replayed steps are whole steps: nothing is left open
  c->mirror_stale = false;
  return MURMUR_OK;
}

murmur_status_t murmur_get_last_error(murmur_cache_t* c, int32_t* device_err_out, void* stream) {
  if (!c || !device_err_out) return MURMUR_ERR_INVALID_ARG;
  MM_CUDA(c, cudaStreamSynchronize((cudaStream_t)stream));
  MM_CUDA(c, cudaMemcpy(device_err_out, c->view.ctrl + kCtrlError, 4, cudaMemcpyDeviceToHost));
  return MURMUR_OK;
}

#ifdef MURMUR_TRACE
murmur_status_t murmur_debug_attn_timeline(murmur_cache_t* c, uint64_t* out, int32_t cap_ctas, int32_t* n_out,
                                           void* stream) {
  if (!c || !n_out || cap_ctas < 0 || (cap_ctas > 0 && !out)) return MURMUR_ERR_INVALID_ARG;
  const int n = c->stats.attn_variant == MURMUR_ATTN_MMA ? c->stats.attn_grid : 0;
  *n_out = n;
  if (n > cap_ctas) return MURMUR_ERR_INVALID_ARG;
  MM_CUDA(c, cudaStreamSynchronize((cudaStream_t)stream));
  if (n > 0)
    MM_CUDA(c, cudaMemcpy(out, c->view.timeline, (size_t)n * kTimelineWords * 8, cudaMemcpyDeviceToHost));
  return MURMUR_OK;
}

murmur_status_t murmur_debug_step_trace(murmur_cache_t* c, uint64_t* out16, void* stream) {
  if (!c || !out16) return MURMUR_ERR_INVALID_ARG;
  MM_CUDA(c, cudaStreamSynchronize((cudaStream_t)stream));
  MM_CUDA(c, cudaMemcpy(out16, c->view.timeline + (size_t)kMaxAttnGrid * kTimelineWords, kStepTraceWords * 8,
                        cudaMemcpyDeviceToHost));
  return MURMUR_OK;
}
#endif  // MURMUR_TRACE

murmur_status_t murmur_set_option(murmur_cache_t* c, int32_t option, int32_t value) {
  if (!c) return MURMUR_ERR_INVALID_ARG;
  switch (option) {
    case MURMUR_OPT_ATTN_VARIANT:
      if (value < MURMUR_ATTN_AUTO || value > MURMUR_ATTN_MMA) return MURMUR_ERR_INVALID_ARG;
      c->attn_variant_opt = value;
      return MURMUR_OK;
    case MURMUR_OPT_ATTN_GRID:
      if (value < 0 || value > kMaxAttnGrid) return MURMUR_ERR_INVALID_ARG;
      c->attn_grid_opt = value;
      return MURMUR_OK;
    case MURMUR_OPT_PDL:
      c->pdl_opt = value != 0;
      return MURMUR_OK;
    case MURMUR_OPT_FUSE_STEP:
      if (value < 0 || value > 2) return MURMUR_ERR_INVALID_ARG;
      c->fuse_step_opt = value;
      return MURMUR_OK;
    case MURMUR_OPT_HOST_ZERO_COPY:
      c->host_zero_copy_opt = value != 0;
      return MURMUR_OK;
    case MURMUR_OPT_L2_KEEP_PCT:
      if (value < -1 || value > 100) return MURMUR_ERR_INVALID_ARG;
      c->l2_keep_pct_opt = value;
      return MURMUR_OK;
    case MURMUR_OPT_PREFILL_VARIANT:
      if (value < MURMUR_PREFILL_AUTO || value > MURMUR_PREFILL_UMMA) return MURMUR_ERR_INVALID_ARG;
      c->prefill_variant_opt = value;
      return MURMUR_OK;
    default:
      return MURMUR_ERR_INVALID_ARG;
  }
}

murmur_status_t murmur_get_stats(murmur_cache_t* c, murmur_stats_t* out) {
  if (!c || !out) return MURMUR_ERR_INVALID_ARG;
  *out = c->stats;
  return MURMUR_OK;
}

murmur_status_t murmur_reset_stats(murmur_cache_t* c) {
  if (!c) return MURMUR_ERR_INVALID_ARG;
  c->stats.kernel_launches = 0;
  c->stats.append_calls = c->stats.evict_calls = c->stats.attn_calls = 0;
  c->stats.host_zero_copy_steps = 0;
  return MURMUR_OK;
}

const char* murmur_last_cuda_error(murmur_cache_t* c) { return c ? cudaGetErrorString(c->last_cuda) : "null handle"; }

const char* murmur_status_str(murmur_status_t s) {
  switch (s) {
    case MURMUR_OK: return "MURMUR_OK";
    case MURMUR_ERR_INVALID_ARG: return "MURMUR_ERR_INVALID_ARG";
    case MURMUR_ERR_STATE: return "MURMUR_ERR_STATE";
    case MURMUR_ERR_OOM_PAGES: return "MURMUR_ERR_OOM_PAGES";
    case MURMUR_ERR_CUDA: return "MURMUR_ERR_CUDA";
    case MURMUR_ERR_UNSUPPORTED: return "MURMUR_ERR_UNSUPPORTED";
    case MURMUR_ERR_SCRATCH_LIMIT: return "MURMUR_ERR_SCRATCH_LIMIT";
  }
  return "MURMUR_ERR_?";
}

const char* murmur_version(void) { return "murmur-b200 0.1 (sm_100a)"; }

}  // extern "C"
