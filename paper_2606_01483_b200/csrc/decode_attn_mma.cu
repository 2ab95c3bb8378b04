// murmur_decode_attn and murmur_decode_step, tensor-core split-K kernel for sm_100a.
//
// Eq. 1 for one query token per sequence over the retained set, all layers in
// ONE persistent launch (the path moves only ~20 MB per layer, so per-layer launches could never
// reach the HBM roofline - DESIGN.md "Kernels").  kStep = true runs the whole decode step (append,
// evict, attention) in that one launch.
//
// Work decomposition
//   item  = (layer, sequence, KV head): G query heads (<= 8) share every K/V row.
//   tile  = <= 64 consecutive retained rows of one run (64/p consecutive live pages), generated
//           in the kernel from the sequence's tile table (closed form of the policy) plus one
//           block-table load per page; identical for all layers and heads of a sequence.
//   The flattened tile list (layer, seq, head, tile) is cut into 2 * grid equal contiguous ranges,
//   two per CTA (split-K across the retained length whenever a cut falls inside an item).
// Per CTA: 2 independent halves, each = 1 producer warp + 4 consumer warps + 3 stages of the ring
//   of (K tile, V tile) buffers, working through its own range - so that one half's end-of-item
//   merge overlaps the other half's streaming - plus, in step mode, one keeper warp.
//   producer : lane j prepares tile j of a batch (pool offsets, sizes), one lane at a time issues
//              1-D bulk copies (cp.async.bulk, TMA engine, L2::evict_first) of each page's
//              contiguous row range straight into the stage buffer; rows are stored pre-swizzled
//              in HBM, so the copy needs no tensor map and ldmatrix is conflict-free.  Bytes
//              copied = retained rows exactly.
//   consumer : the 4 warps of a half take the 4 16-row slices of each tile.  S^T[16 tok x 8 heads]
//              = K Q^T with mma.sync m16n8k16 bf16 (tokens are M, the padded head group is N: 7/8
//              useful), fp32 online softmax in exp2 form, P^T moved to the B-operand layout with
//              movmatrix, O^T[128 d x 8 heads] += V^T P^T with ldmatrix.trans.
//   merge    : at the end of an item the 4 warps' (m, l, O^T) are tree-merged in the MMA fragment
//              layout through shared memory (only the receiving warp waits); the half's first warp
//              writes the output, or - for an item that spans several ranges - publishes a partial
//              and, if it is the LAST contributor (arrival counter), merges all of them.
//   keeper   : step mode only - row scatter k_new/v_new -> pools, the eviction's table products,
//              and (last CTA through a ticket) the integer commit + freeing of dead pages.
#include <cuda_bf16.h>

#include "evict_body.cuh"
#include "ptx_utils.cuh"

namespace murmur {
namespace {

constexpr int kStages = 6;
constexpr int kMinTilesPerRange = 6;
constexpr int kSliceWarps = 4;   // the four 16-row slices of a 64-row tile, one warp each
constexpr int kGroups = 2;       // warp groups; each works through its OWN tile range, fed through its own half of the ring
constexpr int kConsumerWarps = kSliceWarps * kGroups;
static_assert(kStages % kGroups == 0, "each group owns kStages / kGroups stages of the ring");
constexpr int kSub = kStages / kGroups;  // stages per group: group g owns stages g, g + kGroups, ...
static_assert(kTileRows == kSliceWarps * 16, "one m16 slice per warp");
constexpr int kConsumerThreads = kConsumerWarps * 32;
constexpr int kMmaThreads = kConsumerThreads + kGroups * 32;  // + one producer warp per group
constexpr int kTileBytes = kTileRows * kRowBytes;            // 16 KB per K or V tile
constexpr int kQBytes = kMaxGroup * kRowBytes;               // 2 KB
constexpr int kFragFloats = 36 * 32;                         // o[32] + m[2] + l[2] per lane, [reg][lane]
static_assert(kFragFloats == kPartialFloats, "split-K partials are stored in the fragment layout");

struct __align__(128) SmemLayout {
  uint8_t kv[kStages][2][kTileBytes];
  uint8_t q[kGroups][2][kQBytes];
  // step mode: this step's K row and V row of the current item (natural layout).  Processed as a
  // 16-row tile of which only row 0 is valid; the rows "behind" it are whatever follows in shared
  // memory (masked), so this must stay in front of a >= 4 KB member.
  uint8_t newrow[kGroups][2][2][kRowBytes];
  float scratch[kGroups][2][kFragFloats];  // per group: two hand-over buffers of the end-of-item tree merge
  unsigned long long full_k[kStages], full_v[kStages], empty[kStages], q_full[kGroups][2], q_empty[kGroups][2];
  int meta[kStages][2];  // row_begin, row_end of the tile in each stage
  int pre[kMaxSeqsAttn + 1];     // tiles of the sequences before each one (exclusive prefix sum of tg[].n_tiles)
  // per-sequence state the tiles are generated from (the kernel does not read the evict's tile list); kept
  // small - 64 sequences have to fit next to the 6-stage ring
  int len[kMaxSeqsAttn];         // length as attended; step mode: AFTER this step's append
  TileGen tg[kMaxSeqsAttn];      // runs + tile offsets of each sequence (closed form of the policy at that length)
  int old_nblk[kMaxSeqsAttn];    // blocks mapped in the block table when the kernel starts
  int newpage[kMaxSeqsAttn];     // step mode: page this step's append maps for the new block, else -1
  uint8_t newatt[kMaxSeqsAttn];  // step mode: bit 0 = this step's token is in the retained set; bit 1 = the tile
                                 // table at this length was found ready (an evict / a step ran at length - 1)
  int tokpage[kMaxSeqsAttn];     // step mode: page this step's token is written to (read BEFORE the ticket: the
                                 // eviction of the same step may unmap that very block)
  int blk_total;                      // step mode: pages this step's append pops
  int abort;
  int chain_ok;                       // step mode: the predecessor's integer state was seen complete before it ended
};
static_assert(sizeof(SmemLayout) <= 227 * 1024, "shared memory budget");

// Named barriers of one consumer group (4 warps): ids 2 + 4 g + k.  sync = wait for `count` threads,
// arrive = count towards it without waiting.
__device__ __forceinline__ void group_sync(int id, int count) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(count) : "memory"); }
__device__ __forceinline__ void group_arrive(int id, int count) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(count) : "memory"); }

// ---- walking the flattened (layer, seq, head, tile) list ---------------------------------------------
struct Cursor {
  int layer, i, h, k;  // layer index inside the call, index into the sequence list, KV head, tile
};

// 32-bit arithmetic throughout: this runs once per range on the kernel's start-up path, where a
// 64-bit division costs ~0.2 us (the launcher rejects problems with >= 2^31 tiles).
__device__ __forceinline__ Cursor locate(const SmemLayout& s, int n_seqs, int n_kv, long long x64) {
  const unsigned x = (unsigned)x64;
  const unsigned per_layer = (unsigned)n_kv * (unsigned)s.pre[n_seqs];
  Cursor c;
  const unsigned layer = x / per_layer;
  unsigned rem = x - layer * per_layer;
  int i = 0;
  while (i + 1 < n_seqs && (unsigned)n_kv * (unsigned)s.pre[i + 1] <= rem) ++i;
  rem -= (unsigned)n_kv * (unsigned)s.pre[i];
  const unsigned h = rem / (unsigned)s.tg[i].n_tiles;
  c.layer = (int)layer;
  c.i = i;
  c.h = (int)h;
  c.k = (int)(rem - h * (unsigned)s.tg[i].n_tiles);
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
  } while (s.tg[c.i].n_tiles == 0);
}

struct AttnParams {
  const uint16_t* q;
  uint16_t* out;
  float* lse;
  const uint16_t* k_new;  // step mode: [n_layers][n_seqs][n_kv][128] rows of this step's token
  const uint16_t* v_new;
  int write_only;         // step mode, layers after the first of a step issued in layer ranges: the integer state is
                          // already committed (slot reserved, eviction done) - only write this range's rows + attend
  int chain;              // step mode: the previous launch of the stream was a step launch of this handle ...
  unsigned chain_expect;  // ... and kCtrlStepDone reads this once all of its keeper warps are done
  int has_window;         // murmur_decode_attn_windowed: attend over the A(t) of THIS policy instead of the sequence's
  int w_s, d, k_s, w_o, k_o;
  int seq_base, n_seqs_total, layer_begin, n_layers_call;
  float sm_scale;
};

// Block -> page for tile generation: blocks below old_nblk are in the table; the one block a decode
// step may add (step mode) is the page the append pops for this sequence.
struct AttnLookup {
  const int32_t* tab;
  int old_nblk, newpage;
  __device__ __forceinline__ int operator()(int b) const { return b < old_nblk ? tab[b] : newpage; }
};

// Exclusive scan over <= 128 values held 4 per lane by one warp; returns the grand total.
// Exclusive scan over <= 32 values, one per lane; returns the grand total.
__device__ __forceinline__ int warp_scan(int v, int& excl, int lane) {
  int inc = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int t = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += t;
  }
  excl = inc - v;
  return __shfl_sync(0xffffffffu, inc, 31);
}
static_assert(kMaxSeqsAttn <= 64, "two sequences per lane in the set-up scans");
// Exclusive scan over <= 64 values held two per lane (v0 = element 2 lane, v1 = element 2 lane + 1).
__device__ __forceinline__ int warp_scan2(int v0, int v1, int& ex0, int& ex1, int lane) {
  int ex;
  const int total = warp_scan(v0 + v1, ex, lane);
  ex0 = ex;
  ex1 = ex + v0;
  return total;
}

// kStep = false: murmur_decode_attn (the cache is as murmur_kv_evict left it).
// kStep = true : the whole decode step in this one launch (murmur_decode_step): every CTA derives
//   the post-append state itself (lengths + 1, the page a new block gets), attends over it with the
//   newest token's K/V rows taken straight from k_new / v_new, while one extra "keeper" warp per
//   CTA scatters those rows into the pools and runs the eviction's table products; the keeper of
//   the last CTA through a ticket commits the integer state and frees the dead pages.
template <bool kStep>
__global__ void __launch_bounds__(kMmaThreads + (kStep ? 32 : 0), 1)
attn_mma_kernel(const __grid_constant__ CacheView c, const __grid_constant__ SeqList list,
                const __grid_constant__ AttnParams prm) {
  extern __shared__ __align__(128) uint8_t smem_raw[];
  SmemLayout& s = *reinterpret_cast<SmemLayout*>(smem_raw);
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int n_threads = kMmaThreads + (kStep ? 32 : 0);
  const int n_seqs = list.n, n_kv = c.n_kv, G = c.group;
  const int p = c.p, plog = c.p_log2;
#ifdef MURMUR_TRACE
  unsigned long long* trace = c.timeline + (size_t)blockIdx.x * kTimelineWords;
  const unsigned long long t_entry = globaltimer_ns();
#endif
  pdl_launch_dependents();

  // ---- setup: barriers, zeroed padding rows of the Q buffers ---------------------------------------
  if (tid == 0) {
    for (int i = 0; i < kStages; ++i) {
      mbar_init(&s.full_k[i], 1);
      mbar_init(&s.full_v[i], 1);
      mbar_init(&s.empty[i], kSliceWarps);
    }
    for (int i = 0; i < 2 * kGroups; ++i) {
      mbar_init(&s.q_full[0][0] + i, 1);
      mbar_init(&s.q_empty[0][0] + i, kSliceWarps);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    s.abort = 0;
    s.blk_total = 0;
  }
  for (int i = tid; i < kGroups * 2 * kQBytes / 4; i += n_threads) reinterpret_cast<uint32_t*>(&s.q[0][0][0])[i] = 0u;
  __syncthreads();
  // Everything above touches only this CTA's shared memory; from here on the kernel reads what
  // earlier kernels of the stream wrote and writes buffers the previous launch may still use.
  //
  // Chained steps.  When the previous launch of the stream was a step launch of this handle, waiting for it to
  // END (griddepcontrol.wait: all its CTAs done and flushed) would leave HBM idle through its tail, the flush
  // and this launch's set-up.  But everything this launch READS - lengths, tile tables, block tables, the free
  // stack, the rows the previous step appended - is final as soon as all of the previous launch's KEEPER warps
  // are done, which is early in that launch: every keeper adds 1 to kCtrlStepDone when it is (release), and
  // this CTA starts reading when the counter reaches the value the host expects (acquire).  Set-up, tile
  // generation, the K/V stream and the products run ahead; every WRITE this launch makes (output, split-K
  // partials and counters, the keepers' scatter / commit / evict) still sits behind griddepcontrol.wait.  The
  // counter is only a go-ahead: if it does not show the expected value in time (a replayed CUDA graph, whose
  // launches the host did not count), the CTA falls back to griddepcontrol.wait, which is always sufficient.
  // The test is "expected <= counter < expected + this launch's own CTAs" (wrap-safe), not equality: keepers of
  // THIS launch add to the same counter, and a CTA that starts after some of them are done - a second-wave CTA when
  // the grid exceeds the SM count, or one delayed by other work - would never see the exact value and spin out the
  // whole time-out with the step's commit and eviction stalled behind it.  A keeper of this launch can only finish
  // after griddepcontrol.wait, i.e. after the predecessor ended, so counter >= expected still means that every
  // keeper of the predecessor is done; every CTA of a launch adds exactly 1, which bounds the window from above.
  bool chained = false;
  if (kStep && prm.chain) {
    if (tid == 0) {
      int ok = 0;
      for (int it = 0; it < 4096 && !ok; ++it) {
        ok = ((unsigned)ld_acquire(&c.ctrl[kCtrlStepDone]) - prm.chain_expect < gridDim.x) ? 1 : 0;
        if (!ok) __nanosleep(64);
      }
      s.chain_ok = ok;
    }
    __syncthreads();
    chained = s.chain_ok != 0;
  }
  if (!chained) pdl_wait();
#ifdef MURMUR_TRACE
  if (tid == 0) {
    trace[0] = globaltimer_ns();
    trace[1] = 0ull;
    trace[2] = smid();
    trace[3] = 0ull;
    trace[4] = t_entry;
    trace[5] = trace[6] = trace[7] = 0ull;
  }
#endif
  // ---- per-sequence state: policy + length -> tile count; step mode: the length after this step ----
  const int free_top = kStep ? c.ctrl[kCtrlFreeTop] : 0;
  for (int i = tid; i < n_seqs; i += n_threads) {
    const SeqDev& sd = c.seqs[list.ids[i]];
    SeqParams sp = load_params(sd);
    const int old_nblk = (sp.len + p - 1) >> plog;
    if (kStep && !prm.write_only) {
      sp.len += 1;
      if (!sd.active || ((sp.len + p - 1) >> plog) > c.max_blocks) s.abort = 2;
    } else if (kStep && (!sd.active || sp.len < 1)) {
      s.abort = 2;
    }
    s.len[i] = sp.len;
    s.old_nblk[i] = old_nblk;
    s.newpage[i] = -1;
    if (kStep) {
      const int xb = (sp.len - 1) >> plog;
      s.tokpage[i] = xb < old_nblk ? c.block_table[(size_t)list.ids[i] * c.max_blocks + xb] : -1;
    }
    bool tg_ready = false;
    // the tile table at this length was written by the last evict / decode step (SeqDev.tg);
    // generate it here only if it is missing (e.g. a bulk append that was not followed by an evict)
    if (!kStep && prm.has_window) {  // per-call window (e.g. per-layer windows): tables generated here
      sp.w_s = prm.w_s; sp.d = prm.d; sp.k_s = prm.k_s; sp.w_o = prm.w_o; sp.k_o = prm.k_o;
      s.tg[i] = make_tilegen(sp, p, plog);
    } else if (ld_acquire(&sd.tg_len[sp.len & 1]) == sp.len) {  // the length validates the table stored before it
      s.tg[i] = sd.tg[sp.len & 1];
      tg_ready = true;
    } else {
      s.tg[i] = make_tilegen(sp, p, plog);
    }
    int last_b = 0;
#pragma unroll
    for (int k = 0; k < 6; ++k)
      if (s.tg[i].rr.mask >> k & 1u) last_b = max(last_b, s.tg[i].rr.b[k]);
    s.newatt[i] = (uint8_t)(((kStep && last_b == sp.len) ? 1 : 0) | (tg_ready ? 2 : 0));
  }
  __syncthreads();
  if (warp == 0) {  // prefix sums over <= 64 sequences (two per lane): tiles, and (step mode) new-block demand
    const int i0 = 2 * lane, i1 = 2 * lane + 1;
    int e0, e1;
    const int tiles_all = warp_scan2(i0 < n_seqs ? s.tg[i0].n_tiles : 0, i1 < n_seqs ? s.tg[i1].n_tiles : 0, e0, e1, lane);
    if (i0 < n_seqs) s.pre[i0] = e0;
    if (i1 < n_seqs) s.pre[i1] = e1;
    if (lane == 0) s.pre[n_seqs] = tiles_all;
    if (kStep) {
      const int need0 = (i0 < n_seqs && ((s.len[i0] + p - 1) >> plog) > s.old_nblk[i0]) ? 1 : 0;
      const int need1 = (i1 < n_seqs && ((s.len[i1] + p - 1) >> plog) > s.old_nblk[i1]) ? 1 : 0;
      const int blk_all = warp_scan2(need0, need1, e0, e1, lane);
      if (blk_all > free_top) {  // cannot happen after the host-side check; all CTAs agree
        if (lane == 0) s.abort = 3;
      } else {  // pops in call order (C3)
        if (need0) {
          const int pg = c.free_stack[free_top - 1 - e0];
          s.newpage[i0] = pg;
          s.tokpage[i0] = pg;
        }
        if (need1) {
          const int pg = c.free_stack[free_top - 1 - e1];
          s.newpage[i1] = pg;
          s.tokpage[i1] = pg;
        }
      }
      if (lane == 0) s.blk_total = blk_all;
    }
  }
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");  // zeroed Q rows vs later bulk copies
  __syncthreads();
  if (s.abort) {
    if (tid == 0) {
      pdl_wait();
      atomicCAS(&c.ctrl[kCtrlError], 0, s.abort);
      if (kStep) atomicAdd(&c.ctrl[kCtrlStepDone], 1);  // a successor must not wait for a keeper that never runs
    }
    return;
  }

  const uint8_t* kpool = reinterpret_cast<const uint8_t*>(c.k_pool);
  const uint8_t* vpool = reinterpret_cast<const uint8_t*>(c.v_pool);
#ifdef MURMUR_TRACE
  if (tid == 0) trace[5] = globaltimer_ns();
#endif

  if (kStep && warp == kConsumerWarps + kGroups) {
    // ===================================== keeper warp =====================================
    // All the old state this CTA needs is in shared memory now: take the ticket first.
    // (write-only layer ranges change no integer state: no ticket, no table products, no commit)
    const bool wo = prm.write_only != 0;
    // Chained launch: the predecessor is still running, but all of ITS keepers are done, so nothing of it reads
    // SeqDev / the table products / the ticket any more (its warps work from shared memory and, lazily, from
    // block-table entries of blocks that are live at its length).  What may run before griddepcontrol.wait is
    // therefore: the table products, the ticket and the commit (a new block-table entry the predecessor never
    // looks at).  What must wait for its end: unmapping + pushing the pages that die at THIS length (the
    // predecessor may still stream them), and everything that reads this call's inputs - k_new / v_new may have
    // been produced by other work of the stream, which only griddepcontrol.wait orders before us.
    // (1) the eviction's table products for the post-append state, spread over the CTAs
    for (int task = (int)blockIdx.x; task < (wo ? 0 : 2 * n_seqs); task += (int)gridDim.x) {
      const int role = 1 + task / n_seqs, i = task % n_seqs;
      const AttnLookup lk{c.block_table + (size_t)list.ids[i] * c.max_blocks, s.old_nblk[i], s.newpage[i]};
      SeqParams sp = load_params(c.seqs[list.ids[i]]);  // regions and policy never change during a step;
      sp.len = s.len[i];                                 // the length (committed at some point of this launch) is ours
      evict_task(c, list.ids[i], sp, role, lk);
    }
    int last = 0;
    if (lane == 0 && !wo) last = (atomicAdd(&c.ctrl[kCtrlAppendTicket], 1) == (int)gridDim.x - 1);
    last = __shfl_sync(0xffffffffu, last, 0);
    // (2) last CTA through the ticket (every CTA has its old state in shared memory by now): commit the append and
    // look up the pages that die at this length.  Sequences whose tile table was found ready (newatt bit 1: an
    // evict or a step ran at length - 1 and freed everything dead THERE) only need the blocks that are dead now
    // and were not then - one or two per step; lane j takes sequences 2 j and 2 j + 1, all loads in flight at once.
    FreeCand fc0, fc1;
    bool fast = true;
    if (last) {
      for (int i = lane; i < n_seqs; i += 32) {
        c.seqs[list.ids[i]].len = s.len[i];
        if (s.newpage[i] >= 0) c.block_table[(size_t)list.ids[i] * c.max_blocks + s.old_nblk[i]] = s.newpage[i];
      }
      if (lane == 0) c.ctrl[kCtrlAppendTicket] = 0;
      const bool ok0 = free_candidates(c, list.ids, n_seqs, 2 * lane, s.len, s.newatt, s.old_nblk, s.newpage, fc0);
      const bool ok1 = free_candidates(c, list.ids, n_seqs, 2 * lane + 1, s.len, s.newatt, s.old_nblk, s.newpage, fc1);
      fast = __all_sync(0xffffffffu, ok0 && ok1);
    }
    if (chained) pdl_wait();
#ifdef MURMUR_TRACE
    if (lane == 0) trace[6] = globaltimer_ns();
#endif
    // (3) this step's K/V rows into the pools: one half-warp per 256-byte row (pre-swizzled), four rows in flight
    {
      const int half = lane >> 4, sub = lane & 15;
      const unsigned per_kv = (unsigned)prm.n_layers_call * (unsigned)n_seqs * (unsigned)n_kv;
      const unsigned stride = 2u * gridDim.x;
      for (unsigned u0 = 2u * blockIdx.x + half; u0 < 2u * per_kv; u0 += 4u * stride) {
        uint4 val[4];
        uint4* dst[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          const unsigned u = u0 + (unsigned)k * stride;
          dst[k] = nullptr;
          if (u >= 2u * per_kv) continue;
          const unsigned is_v = u >= per_kv, r = is_v ? u - per_kv : u;
          const unsigned r2 = r / (unsigned)n_kv, h = r - r2 * (unsigned)n_kv;
          const unsigned lc = r2 / (unsigned)n_seqs, i = r2 - lc * (unsigned)n_seqs;
          const int slot = (s.len[i] - 1) & (p - 1);
          const int page = s.tokpage[i];
          if (page < 0) {
            // write-only range: the eviction of this step (run with the first range) may already have
            // freed the block of a token that is dead on arrival (w_out = 0) - its rows are dropped
            if (!(wo && !(s.newatt[i] & 1))) atomicCAS(&c.ctrl[kCtrlError], 0, 2);
            continue;
          }
          val[k] = reinterpret_cast<const uint4*>(is_v ? prm.v_new : prm.k_new)[(size_t)r * 16 + sub];
          uint8_t* pool = reinterpret_cast<uint8_t*>(is_v ? c.v_pool : c.k_pool);
          dst[k] = reinterpret_cast<uint4*>(pool + row_offset(c, prm.layer_begin + (int)lc, page, (int)h, slot)) + (sub ^ (slot & 7));
        }
#pragma unroll
        for (int k = 0; k < 4; ++k)
          if (dst[k] != nullptr) *dst[k] = val[k];
      }
    }
    // (4) last keeper: push + unmap the dead pages (sequences in call order, blocks ascending - DESIGN.md C3)
    if (last) {
      const int top0 = free_top - s.blk_total;
      if (fast) {
        int e0, e1;
        const int total_free = warp_scan2(fc0.n, fc1.n, e0, e1, lane);
        free_push(c, list.ids, 2 * lane, fc0, top0 + e0);
        free_push(c, list.ids, 2 * lane + 1, fc1, top0 + e1);
        if (lane == 0) c.ctrl[kCtrlFreeTop] = top0 + total_free;
      } else {
        __syncwarp();
        evict_free_warp(c, list.ids, n_seqs, s.len, top0);
      }
    }
    __threadfence();  // release: this keeper's table products, rows and (last keeper) commit + freed pages ...
    asm volatile("fence.proxy.async;" ::: "memory");  // (the successor reads the scattered rows with bulk copies)
    __syncwarp();
    if (lane == 0) atomicAdd(&c.ctrl[kCtrlStepDone], 1);  // ... before the count a chained successor waits for
#ifdef MURMUR_TRACE
    if (lane == 0) trace[7] = globaltimer_ns();
#endif
    return;
  }

  // Work split: the flattened (layer, seq, head, tile) list is cut into V equal contiguous ranges,
  // two per CTA - one per consumer group (split-K wherever a cut falls inside an item).  The two
  // groups of a CTA work through their ranges independently, each fed through its own half of the
  // ring: while one group is in its end-of-item merge (~2 us, no tiles consumed) the other keeps
  // streaming, so the merges no longer stall the CTA's share of HBM.
  const long long total = (long long)prm.n_layers_call * n_kv * s.pre[n_seqs];
  if (total > 0x7fffffffLL) {  // the range arithmetic below is 32-bit (2^31 tiles = 64 TB of K/V per launch)
    if (tid == 0) atomicCAS(&c.ctrl[kCtrlError], 0, 5);
    return;
  }
  // Number of ranges: two per CTA, but never fewer than kMinTilesPerRange tiles each - a launch with little work
  // (one layer of a layer-by-layer engine: a few hundred tiles) would otherwise cut every item into many
  // one- or two-tile segments, each paying a Q load, a tree merge and a split-K partial.  Range v belongs to
  // half v / gridDim.x of CTA v % gridDim.x, so a short range list is spread over all SMs first.
  const long long V = max(1ll, min(min(total, (long long)kGroups * gridDim.x), total / kMinTilesPerRange));
  if ((long long)blockIdx.x >= V) return;
  // range v = [v total / V, (v + 1) total / V), in 32-bit arithmetic (v r < V^2 <= 2^22)
  const unsigned rq = (unsigned)total / (unsigned)V, rr = (unsigned)total - rq * (unsigned)V;
  auto range_lo = [&](long long v) { return (long long)((unsigned)v * rq + ((unsigned)v * rr) / (unsigned)V); };
  if (warp >= kConsumerWarps) {
    // ================================ producer warps (one per group) ================================
    const int gg = warp - kConsumerWarps;
    // Walks its tile range in batches of <= 32 tiles of one item; lane j owns tile j of the batch.
    // Everything a tile's copies need (pool offsets, sizes, destination rows) is computed by all
    // lanes in parallel, right after the previous batch has been issued (the ring is full then, so
    // the table loads hide behind it), from the sequence's tile table plus one block-table load
    // per page - so the serial part of issuing a tile (one lane at a time, ring order) is only:
    // wait for the stage, 2 expect_tx, the copies.  That serial path runs at single-warp latency
    // and has to stay well below the ~0.75 us a tile takes to stream at this CTA's share of HBM.
    const unsigned long long kv_policy = c.l2_keep > 0.f ? l2_policy_keep_fraction(c.l2_keep) : l2_policy_evict_first();
    struct TileIssue {
      unsigned long long off[4];  // byte offset of the page's first copied row in a pool (same in K and V)
      uint32_t dst[4], bytes[4];  // destination offset in the stage buffer, bytes to copy (0 = none)
      int row_begin, row_end;     // valid rows of the tile buffer
      uint32_t tx;                // bytes arriving through bulk copies, per K / V barrier
    };
    auto prep = [&](const Cursor& cc, int tix) {
      const AttnLookup lk{c.block_table + (size_t)list.ids[cc.i] * c.max_blocks, s.old_nblk[cc.i], s.newpage[cc.i]};
      const TileDesc td = tile_at(s.tg[cc.i], tix, p, plog, lk);
      TileIssue ti;
      ti.row_begin = td.row_begin;
      ti.row_end = td.row_end;
      // step mode: this step's token (if attended) is the last row of the item's last tile; it is not
      // in the pool yet and is handled apart (newrow), so the tile ends one row earlier
      const int row_end_pool = td.row_end - ((kStep && (s.newatt[cc.i] & 1) && tix == s.tg[cc.i].n_tiles - 1) ? 1 : 0);
      ti.row_end = row_end_pool;
      ti.tx = (uint32_t)(row_end_pool - td.row_begin) * kRowBytes;
      const int layer = prm.layer_begin + cc.layer;
#pragma unroll
      for (int pg = 0; pg < 4; ++pg) {
        const int r0 = (pg == 0) ? td.row_begin : pg * p;
        const int r1 = (pg == td.n_pages - 1) ? row_end_pool : (pg + 1) * p;
        const bool on = pg < td.n_pages && r1 > r0;
        ti.off[pg] = on ? row_offset(c, layer, td.page[pg], cc.h, r0 - pg * p) : 0ull;
        ti.dst[pg] = (uint32_t)r0 * kRowBytes;
        ti.bytes[pg] = on ? (uint32_t)(r1 - r0) * kRowBytes : 0u;
      }
      return ti;
    };
    // This producer warp feeds consumer group gg: it walks the group's range in batches of <= 32
    // tiles of one item; lane j of the warp holds the prepared copies of tile j of the batch.
    const long long v = (long long)gg * gridDim.x + blockIdx.x;
    if (v >= V) return;
    const long long lo = range_lo(v), hi = range_lo(v + 1);
    Cursor cur = locate(s, n_seqs, n_kv, lo);
    long long remaining = hi - lo;  // tiles left, counted from the start of the current item's segment
    int seg = (int)min((long long)(s.tg[cur.i].n_tiles - cur.k), remaining);
    int base = 0, cnt = min(32, seg);
    int sub = 0;         // position of the next tile in the group's kSub stages
    uint32_t ph = 0;     // its phase parity
    int item_no = 0;
    TileIssue ti;
    if (lane < cnt) ti = prep(cur, cur.k + lane);
    while (remaining > 0) {
      // ---- issue the current batch ----
      // first batch of an item (or of this range's segment of it): stage its G query rows and, in step mode, this
      // step's K / V rows of the item when this segment ends with the item's last tile (natural layout, straight
      // from k_new / v_new).  These are the call's INPUTS: in a chained launch they are read only after
      // griddepcontrol.wait (other work of the stream may have produced them) - for the first item that wait is
      // put off until the ring is full, so the K/V stream starts while the predecessor drains.
      auto load_q = [&]() {
        if (kStep && chained) pdl_wait();
        const int qb = item_no & 1;
        mbar_wait(&s.q_empty[gg][qb], ((item_no >> 1) & 1) ^ 1);
        const bool mini = kStep && (s.newatt[cur.i] & 1) && (cur.k + seg == s.tg[cur.i].n_tiles);
        const size_t seq_row = (size_t)cur.layer * prm.n_seqs_total + prm.seq_base + cur.i;
        mbar_expect_tx(&s.q_full[gg][qb], (uint32_t)((G + (mini ? 2 : 0)) * kRowBytes));
        bulk_g2s(&s.q[gg][qb][0], prm.q + (seq_row * c.n_q + (size_t)cur.h * G) * kHeadDim, (uint32_t)(G * kRowBytes),
                 &s.q_full[gg][qb]);
        if (mini) {
          const size_t off = (seq_row * n_kv + cur.h) * kHeadDim;
          bulk_g2s(&s.newrow[gg][qb][0][0], prm.k_new + off, (uint32_t)kRowBytes, &s.q_full[gg][qb]);
          bulk_g2s(&s.newrow[gg][qb][1][0], prm.v_new + off, (uint32_t)kRowBytes, &s.q_full[gg][qb]);
        }
      };
      const bool first_batch = base == 0 && lane == 0;
      const bool defer_q = kStep && chained && item_no == 0;
      if (first_batch && !defer_q) load_q();
      for (int j = 0; j < cnt; ++j) {
        const int st = kGroups * sub + gg;
        if (first_batch && defer_q && j == kSub) load_q();  // the ring is full: tile j needs a stage back
        if (lane == j) {
          mbar_wait(&s.empty[st], ph ^ 1u);
          s.meta[st][0] = ti.row_begin;
          s.meta[st][1] = ti.row_end;
          mbar_expect_tx(&s.full_k[st], ti.tx);  // 0 bytes (a tile that held only the new row) = plain arrive
          mbar_expect_tx(&s.full_v[st], ti.tx);
#pragma unroll
          for (int pg = 0; pg < 4; ++pg) {
            if (ti.bytes[pg]) {
              bulk_g2s_hint(&s.kv[st][0][ti.dst[pg]], kpool + ti.off[pg], ti.bytes[pg], &s.full_k[st], kv_policy);
              bulk_g2s_hint(&s.kv[st][1][ti.dst[pg]], vpool + ti.off[pg], ti.bytes[pg], &s.full_v[st], kv_policy);
            }
          }
        }
        __syncwarp();
        if (++sub == kSub) {
          sub = 0;
          ph ^= 1u;
        }
      }
      if (first_batch && defer_q && cnt <= kSub) load_q();
      // ---- advance, and prepare the next batch while the ring (just filled) drains ----
      base += cnt;
      if (base >= seg) {  // item (or this range's segment of it) done
        remaining -= seg;
        base = 0;
        ++item_no;
        if (remaining > 0) {
          next_item(s, n_seqs, n_kv, cur);
          seg = (int)min((long long)s.tg[cur.i].n_tiles, remaining);
        }
      }
      cnt = remaining > 0 ? min(32, seg - base) : 0;
      if (lane < cnt) ti = prep(cur, cur.k + base + lane);
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

  // this group's tile range
  const long long vrange = (long long)grp * gridDim.x + blockIdx.x;
  if (vrange >= V) return;
  const long long lo = range_lo(vrange), hi = range_lo(vrange + 1);
  const int bar0 = 2 + 4 * grp;  // this group's named barriers
  Cursor cur = locate(s, n_seqs, n_kv, lo);
  long long remaining = hi - lo;
  long long pos = lo;
  uint32_t n = 0;  // tiles of this group's stream consumed so far
  int item_no = 0;
  bool first_segment = true;

  while (remaining > 0) {
    const int nt_i = s.tg[cur.i].n_tiles;
    const int seg = (int)min((long long)(nt_i - cur.k), remaining);
    const bool complete = (cur.k == 0) && (seg == nt_i);

    // ---- this item's query fragments (B operand of S^T = K Q^T) ----
    const int qb = item_no & 1;
    mbar_wait(&s.q_full[grp][qb], (item_no >> 1) & 1);
    uint32_t qf[8][2];
    {
      const uint8_t* qs = &s.q[grp][qb][0] + lrow * kRowBytes + lcol * 2;
#pragma unroll
      for (int ks = 0; ks < 8; ++ks) {
        qf[ks][0] = *reinterpret_cast<const uint32_t*>(qs + ks * 32);
        qf[ks][1] = *reinterpret_cast<const uint32_t*>(qs + ks * 32 + 16);
      }
    }
    __syncwarp();
    // step mode: the group's first warp also processes this step's token at the end of the item, from
    // the same double buffer as the queries - it hands the buffer back only then
    const bool mini = kStep && w4 == 0 && (s.newatt[cur.i] & 1) && (cur.k + seg == nt_i);
    if (lane == 0 && !mini) mbar_arrive(&s.q_empty[grp][qb]);

    float m0 = -INFINITY, m1 = -INFINITY, l0 = 0.f, l1 = 0.f;
    float o[8][4];
#pragma unroll
    for (int dt = 0; dt < 8; ++dt) o[dt][0] = o[dt][1] = o[dt][2] = o[dt][3] = 0.f;

    // One 16-row slice of a tile whose K / V buffers start at kbase / vbase (shared-memory
    // addresses of row 0), valid rows [rb, re).  v_ready: barrier the V data arrives on, or null.
    auto slice = [&](uint32_t kbase, uint32_t vbase, int rb, int re, unsigned long long* v_ready, uint32_t ph) {
      const bool act = max(slice0, rb) < min(slice0 + 16, re);  // warp-uniform: the slice holds a valid row (a tile may be empty)
      uint32_t pb0 = 0u, pb1 = 0u;
      if (act) {
        // ---- S^T[16 x 8] = K Q^T, two independent accumulator chains ----
        const uint32_t rowaddr = kbase + k_off;
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
      if (v_ready != nullptr) mbar_wait(v_ready, ph);
      if (act) {
        const uint32_t rowaddr = vbase + v_off;
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
    };

    for (int tt = 0; tt < seg; ++tt) {
      const uint32_t nn = n + (uint32_t)tt;
      const int st = kGroups * (int)(nn % kSub) + grp;
      const uint32_t ph = (nn / kSub) & 1u;
      mbar_wait(&s.full_k[st], ph);
      slice(smem_u32(&s.kv[st][0][0]), smem_u32(&s.kv[st][1][0]), s.meta[st][0], s.meta[st][1], &s.full_v[st], ph);
      __syncwarp();
      if (lane == 0) mbar_arrive(&s.empty[st]);
    }
    if (mini) {  // first warp of the group (slice0 == 0): a tile whose only valid row, row 0, is this step's token
      slice(smem_u32(&s.newrow[grp][qb][0][0]), smem_u32(&s.newrow[grp][qb][1][0]), 0, 1, nullptr, 0u);
      __syncwarp();
      if (lane == 0) mbar_arrive(&s.q_empty[grp][qb]);
    }
    n += (uint32_t)seg;

    // ---- end of the item (or of this range's segment of it): tree merge of the group's four row
    // slices in the MMA fragment layout (lane for lane, no transposition): warps 2, 3 hand their
    // (m, l, O^T) to warps 0, 1, then warp 1 to warp 0.  Only the receiving side waits; a warp that
    // has handed over goes straight on to the next item.
    auto put = [&](float* fs) {
#pragma unroll
      for (int dt = 0; dt < 8; ++dt) {
#pragma unroll
        for (int e = 0; e < 4; ++e) fs[(dt * 4 + e) * 32 + lane] = o[dt][e];
      }
      fs[32 * 32 + lane] = m0;
      fs[33 * 32 + lane] = m1;
      fs[34 * 32 + lane] = l0;
      fs[35 * 32 + lane] = l1;
    };
    // (m, l, O) <- LSE-merge of itself and the fragment at fs (shared or global memory)
    auto take = [&](const float* fs, bool global) {
      auto ld = [&](int r) { return global ? __ldcg(fs + r * 32 + lane) : fs[r * 32 + lane]; };
      const float mo0 = ld(32), mo1 = ld(33);
      const float mn0 = fmaxf(m0, mo0), mn1 = fmaxf(m1, mo1);
      const float fa0 = (m0 == -INFINITY) ? 0.f : ex2((m0 - mn0) * c2);
      const float fa1 = (m1 == -INFINITY) ? 0.f : ex2((m1 - mn1) * c2);
      const float fb0 = (mo0 == -INFINITY) ? 0.f : ex2((mo0 - mn0) * c2);
      const float fb1 = (mo1 == -INFINITY) ? 0.f : ex2((mo1 - mn1) * c2);
      l0 = l0 * fa0 + ld(34) * fb0;
      l1 = l1 * fa1 + ld(35) * fb1;
#pragma unroll
      for (int dt = 0; dt < 8; ++dt) {
        o[dt][0] = o[dt][0] * fa0 + ld(dt * 4 + 0) * fb0;
        o[dt][1] = o[dt][1] * fa1 + ld(dt * 4 + 1) * fb1;
        o[dt][2] = o[dt][2] * fa0 + ld(dt * 4 + 2) * fb0;
        o[dt][3] = o[dt][3] * fa1 + ld(dt * 4 + 3) * fb1;
      }
      m0 = mn0;
      m1 = mn1;
    };
    // all four warps have finished the item's tiles; the hand-over buffers of the previous item are free
    group_sync(bar0 + 0, kSliceWarps * 32);
    if (w4 >= 2) {
      put(s.scratch[grp][w4 - 2]);
      group_arrive(bar0 + 1, kSliceWarps * 32);
    } else {
      group_sync(bar0 + 1, kSliceWarps * 32);
      take(s.scratch[grp][w4], false);
      if (w4 == 1) {
        put(s.scratch[grp][1]);  // warp 1 has just read this buffer itself
        group_arrive(bar0 + 2, 2 * 32);
      } else {
        group_sync(bar0 + 2, 2 * 32);
        take(s.scratch[grp][1], false);
      }
    }

    if (w4 == 0) {
      // ---- the group's first warp finishes the item: output, or split-K partial ----
      if (kStep && chained) pdl_wait();  // first global write of this warp (no-op once the predecessor has ended)
      const int layer_c = cur.layer;
      const size_t out_row0 = ((size_t)layer_c * prm.n_seqs_total + prm.seq_base + cur.i) * c.n_q + (size_t)cur.h * G;
      // lane (lrow, lcol) holds O^T[d][head] for d = 16 dt + lrow (+ 8), head = lcol (+ 1)
      auto write_out = [&]() {
        float t0 = l0, t1 = l1;  // l is still split over the 8 row groups (lrow) of the fragment
#pragma unroll
        for (int sh = 4; sh <= 16; sh <<= 1) {
          t0 += __shfl_xor_sync(0xffffffffu, t0, sh);
          t1 += __shfl_xor_sync(0xffffffffu, t1, sh);
        }
        const float i0 = 1.f / t0, i1 = 1.f / t1;
        uint16_t* o0 = prm.out + (out_row0 + lcol) * kHeadDim;
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
        if (prm.lse != nullptr && lrow == 0) {
          if (lcol < G) prm.lse[out_row0 + lcol] = m0 * prm.sm_scale + __logf(t0);
          if (lcol + 1 < G) prm.lse[out_row0 + lcol + 1] = m1 * prm.sm_scale + __logf(t1);
        }
      };
      if (complete) {
        write_out();
      } else {
        // split item: publish this range's partial (fragment layout); the last contributor merges all.
        // Contributors = the ranges v_first..v_last that intersect the item.
        const long long item_lo = pos - cur.k;
        // range containing tile x = floor(((x + 1) V - 1) / total)
        const long long v_first = ((item_lo + 1) * V - 1) / total;
        const long long v_last = ((item_lo + nt_i) * V - 1) / total;
        float* part = c.partials + (size_t)(2 * vrange + (first_segment ? 0 : 1)) * kPartialFloats;
        put(part);
        __threadfence();  // release: the partial before the ticket
        __syncwarp();
        int* counter = c.item_counters + ((size_t)layer_c * n_seqs + cur.i) * n_kv + cur.h;
        int last = 0;
        if (lane == 0) last = (atomicAdd(counter, 1) == (int)(v_last - v_first));
        last = __shfl_sync(0xffffffffu, last, 0);
        if (last) {
          __threadfence();
          m0 = m1 = -INFINITY;
          l0 = l1 = 0.f;
#pragma unroll
          for (int dt = 0; dt < 8; ++dt) o[dt][0] = o[dt][1] = o[dt][2] = o[dt][3] = 0.f;
          for (long long vv = v_first; vv <= v_last; ++vv) {
            // a contributor used its second slot for this item iff its range starts before the item
            const int sl = 2 * (int)vv + ((range_lo(vv) < item_lo) ? 1 : 0);
            take(c.partials + (size_t)sl * kPartialFloats, true);
          }
          write_out();
          if (lane == 0) *counter = 0;  // self-resetting for the next launch
        }
      }
    }

    remaining -= seg;
    pos += seg;
    first_segment = false;
    ++item_no;
    next_item(s, n_seqs, n_kv, cur);
  }
#ifdef MURMUR_TRACE
  if (w4 == 0 && lane == 0) {
    atomicMax(&trace[1], globaltimer_ns());
    atomicAdd(&trace[3], (unsigned long long)(hi - lo));
  }
#endif
}

}  // namespace

namespace {

template <bool kStep>
cudaError_t launch_mma(const CacheView& c, const SeqList& list, const AttnParams& prm_in, int grid, bool pdl,
                       cudaStream_t st, LaunchInfo* info) {
  const int smem = (int)sizeof(SmemLayout);
  cudaError_t ea = opt_in_smem_once(kStep ? kSmemStep : kSmemAttn, reinterpret_cast<const void*>(attn_mma_kernel<kStep>), smem);
  if (ea != cudaSuccess) return ea;
  if (grid > kMaxAttnGrid) grid = kMaxAttnGrid;
  AttnParams prm = prm_in;
  PdlLaunch l(dim3((unsigned)grid), dim3(kMmaThreads + (kStep ? 32 : 0)), (size_t)smem, st, pdl);
  info->launches += 1;
  info->grid = grid;
  info->smem = smem;
  return cudaLaunchKernelEx(&l.cfg, attn_mma_kernel<kStep>, c, list, prm);
}

}  // namespace

cudaError_t launch_attn_mma(const CacheView& c, const SeqList& list, int seq_base, int n_seqs_total, const void* q,
                            void* out, float* lse, int layer_begin, int layer_end, float sm_scale, int grid,
                            bool pdl, const SeqParams* window, cudaStream_t st, LaunchInfo* info) {
  AttnParams prm{};
  if (window != nullptr) {
    prm.has_window = 1;
    prm.w_s = window->w_s; prm.d = window->d; prm.k_s = window->k_s; prm.w_o = window->w_o; prm.k_o = window->k_o;
  }
  prm.q = reinterpret_cast<const uint16_t*>(q);
  prm.out = reinterpret_cast<uint16_t*>(out);
  prm.lse = lse;
  prm.seq_base = seq_base;
  prm.n_seqs_total = n_seqs_total;
  prm.layer_begin = layer_begin;
  prm.n_layers_call = layer_end - layer_begin;
  prm.sm_scale = sm_scale;
  return launch_mma<false>(c, list, prm, grid, pdl, st, info);
}

// The whole decode step (append one token per sequence, evict, attend) as ONE launch over the layers
// [layer_begin, layer_end); write_only: a later layer range of a step whose first range has already
// reserved the slots and run the eviction.
cudaError_t launch_step_mma(const CacheView& c, const SeqList& list, const void* k_new, const void* v_new,
                            const void* q, void* out, float* lse, float sm_scale, int layer_begin, int layer_end,
                            bool write_only, int grid, bool pdl, long long chain_expect, cudaStream_t st, LaunchInfo* info) {
  AttnParams prm{};
  prm.q = reinterpret_cast<const uint16_t*>(q);
  prm.out = reinterpret_cast<uint16_t*>(out);
  prm.lse = lse;
  prm.k_new = reinterpret_cast<const uint16_t*>(k_new);
  prm.v_new = reinterpret_cast<const uint16_t*>(v_new);
  prm.seq_base = 0;
  prm.n_seqs_total = list.n;
  prm.layer_begin = layer_begin;
  prm.n_layers_call = layer_end - layer_begin;
  prm.write_only = write_only ? 1 : 0;
  prm.chain = (pdl && chain_expect >= 0) ? 1 : 0;
  prm.chain_expect = (unsigned)chain_expect;
  prm.sm_scale = sm_scale;
  return launch_mma<true>(c, list, prm, grid, pdl, st, info);
}

}  // namespace murmur
