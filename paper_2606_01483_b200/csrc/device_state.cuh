// Device-resident state of a murmur cache and the by-value view handed to every kernel.
//
// HBM layout:
//   K pool, V pool : [layer][page][kv_head][slot][128] bf16 - a (layer, page, head) chunk is
//                    page_size * 256 contiguous bytes.  Inside a 256-byte row the sixteen 16-byte
//                    chunks are stored XOR-swizzled by (slot & 7): logical chunk c of slot s sits
//                    at chunk position c ^ (s & 7).  A 1-D bulk copy of any slot range therefore
//                    lands in shared memory already laid out for conflict-free ldmatrix.
//   workspace      : SeqDev[max_seqs] | block_table | live_pages | live_blocks | tiles |
//                    free_stack | ctrl words | item counters | split-K partials | staging
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "policy_math.cuh"

namespace murmur {

constexpr int kHeadDim = 128;
constexpr int kRowBytes = kHeadDim * 2;  // one K or V row of one head
constexpr int kTileRows = 64;            // rows of one attention tile (tokens)
constexpr int kMaxGroup = 8;             // query heads per KV head, padded to the MMA N = 8
constexpr int kMaxRuns = 6;
constexpr int kMaxSeqsPerLaunch = 128;
constexpr int kMaxSeqsAttn = 64;         // sequences per launch of the tensor-core attention kernel (smem tables)
constexpr int kOStride = 132;            // floats per head row in split-K partials / merge scratch
constexpr int kPartialFloats = 36 * 32;   // split-K partial in MMA fragment layout: o[32] + m[2] + l[2] per lane, [reg][lane]
constexpr int kMaxAttnGrid = 1024;       // upper bound on CTAs of the persistent attention kernel
constexpr int kStepTraceWords = 16;      // globaltimer stamps of the step prologue (after the per-CTA entries)
constexpr int kTimelineWords = 8;        // globaltimer at CTA start, at CTA end, SM id, tiles processed; entry, set-up done, keeper begin, keeper end

// ctrl word indices
enum { kCtrlFreeTop = 0, kCtrlError = 1, kCtrlAppendTicket = 2, kCtrlStepDone = 3, kCtrlWords = 8 };

// The maximal intervals of A(t) held in six fixed slots (all indexing static, so the whole thing
// lives in registers): slot i is a run iff bit i of `mask` is set; merged neighbours are folded
// into the lowest slot of their group.
struct Runs6 {
  int32_t a[6], b[6];
  uint32_t mask;
};

// Attention tiles of one sequence, generated from the runs: a tile is <= 64 consecutive rows of
// one run = 64/p consecutive (live) blocks.  toff[i] = tiles before slot i.
struct TileGen {
  Runs6 rr;
  int32_t toff[6];
  int32_t n_tiles, n_ret;
};

struct SeqDev {  // 320 bytes
  int32_t P, S, M, len;
  int32_t w_s, d, k_s, w_o, k_o;
  int32_t active;
  int32_t n_live;      // live (allocated) blocks after the last evict
  int32_t n_runs;      // maximal intervals of the retained set
  int32_t n_tiles;     // attention tiles (tensor-core path)
  int32_t n_retained;  // |A(t)|
  int32_t runs[kMaxRuns][3];  // first_pos, n_tok, index of first block in live list
  // Tile tables of the retained set, double-buffered by length parity: tg[x & 1] is the table at
  // length x iff tg_len[x & 1] == x.  An evict at length L writes the tables for L and L + 1, so
  // the next decode step (which attends at L + 1) finds its table ready and only copies it.
  TileGen tg[2];
  int32_t tg_len[2];
  // indexed mode (kv_indexed.cu): rows stored densely per (layer, KV head) slab; blocks 0 .. idx_blocks-1 mapped
  int32_t idx_mode;      // 1: the sequence is in indexed mode (the positional fields above no longer apply)
  int32_t idx_blocks;    // logical blocks mapped
  int32_t idx_next_pos;  // original position the next appended token gets
  int32_t idx_max_len;   // rows of the longest slab
};
static_assert(sizeof(SeqDev) == 320, "SeqDev must be 320 bytes");

struct __align__(16) TileDesc {  // 32 bytes: one <= 64-row tile of one run, same for all layers/heads
  int32_t page[4];     // physical pages of the tile, in order (unused = -1)
  int32_t row_begin;   // first valid row of the tile buffer (= first slot in page[0])
  int32_t row_end;     // one past the last valid row (rows are page j * p + slot)
  int32_t n_pages;
  int32_t first_pos;   // absolute position of row_begin (debug / profiler use)
};
static_assert(sizeof(TileDesc) == 32, "TileDesc must be 32 bytes");

struct CacheView {
  int32_t n_layers, n_q, n_kv, p, p_log2, max_seqs, max_blocks, group;
  int64_t n_pages;
  uint16_t* k_pool;
  uint16_t* v_pool;
  SeqDev* seqs;
  int32_t* block_table;  // [max_seqs][max_blocks] logical block -> page / -1
  int32_t* live_pages;   // [max_seqs][max_blocks]
  int32_t* live_blocks;  // [max_seqs][max_blocks]
  TileDesc* tiles;       // [max_seqs][max_blocks]
  int32_t* free_stack;   // [n_pages]
  int32_t* ctrl;         // [kCtrlWords]
  int32_t* item_counters;  // [n_layers][max_seqs][n_kv] split-K arrival counters (self-resetting)
  float* partials;       // [4 * kMaxAttnGrid][kPartialFloats]: two slots per tile range, two ranges per CTA
  unsigned long long* timeline;  // [kMaxAttnGrid][kTimelineWords] per-CTA trace of the last attention launch
  float l2_keep;         // fraction of the K/V rows decode attention reads with L2::evict_last (the rest: evict_first)
};

#ifdef __CUDACC__
__device__ __forceinline__ unsigned long long globaltimer_ns() {
  unsigned long long t;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
  return t;
}
// Step-prologue trace (profiling aid): word k of the block behind the per-CTA attention entries.
// 0 append start (CTA 0, after the dependency wait)   1 last append CTA passed the ticket
// 2 commit done   3 evict body start   4 evict body end
// 5.. the last CTA's own phases: 5 after its dependency wait, 6 old state loaded, 7 prefix sums
// done, 8 row loads issued, 9 eviction tasks done, 10 page ids consumed, 11 block index
// Compiled in only with -DMURMUR_TRACE (profiling builds): the production kernels carry no stamps.
__device__ __forceinline__ void step_stamp(const CacheView& c, int k) {
#ifdef MURMUR_TRACE
  c.timeline[(size_t)kMaxAttnGrid * kTimelineWords + k] = globaltimer_ns();
#else
  (void)c; (void)k;
#endif
}
#endif

// Indexed-mode tables, in a caller-provided device buffer (murmur_indexed_enable):
//   len [max_seqs][n_layers * n_kv]        rows of each slab
//   pos [max_seqs][n_layers * n_kv][cap]   original position of the row in each slot (ascending), cap = max_blocks * p
struct IdxView {
  int32_t* len;
  int32_t* pos;
  int32_t cap;
};

struct SeqList {  // per-launch sequence list, passed by value (no H2D copy, graph-capturable)
  int32_t n;
  int32_t ids[kMaxSeqsPerLaunch];
};

struct AppendList {
  int32_t n;
  int32_t ids[kMaxSeqsPerLaunch];
  int32_t n_tok[kMaxSeqsPerLaunch];
};

// Byte offset of row (layer, page, head, slot) in a pool.
__host__ __device__ __forceinline__ size_t row_offset(const CacheView& c, int layer, int page, int head, int slot) {
  return ((((size_t)layer * (size_t)c.n_pages + (size_t)page) * c.n_kv + head) * c.p + slot) * (size_t)kRowBytes;
}

__device__ __forceinline__ SeqParams load_params(const SeqDev& s) {
  SeqParams r;
  r.P = s.P; r.S = s.S; r.M = s.M; r.len = s.len;
  r.w_s = s.w_s; r.d = s.d; r.k_s = s.k_s; r.w_o = s.w_o; r.k_o = s.k_o;
  return r;
}

// ---- programmatic dependent launch (PDL) ------------------------------------------------------
// Every kernel of the decode step starts with pdl_launch_dependents() (the next kernel of the
// stream may become resident and run its prologue) and calls pdl_wait() before its first access
// to memory another kernel of the stream may have written - or may still be reading, for data it
// is about to overwrite.  griddepcontrol.wait returns when ALL prerequisite grids have completed
// and flushed, so the ordering is that of ordinary stream serialisation; only launch latency and
// kernel prologues overlap.  Both are no-ops when the kernel was launched without the attribute.
#ifdef __CUDACC__
// Acquire load (gpu scope): pairs with the writer's __threadfence() before it publishes a flag / length.
__device__ __forceinline__ int32_t ld_acquire(const int32_t* p) {
  int32_t v;
  asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
#endif

// Launch configuration helper: sets the programmatic-stream-serialisation attribute when `pdl`.
struct PdlLaunch {
  cudaLaunchConfig_t cfg;
  cudaLaunchAttribute attr[1];
  PdlLaunch(dim3 grid, dim3 block, size_t smem, cudaStream_t st, bool pdl) {
    cfg = cudaLaunchConfig_t{};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = pdl ? 1 : 0;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
  }
};

// Opt a kernel in to `smem` bytes of dynamic shared memory, once per (kernel, device): the attribute is
// per device, and handles on several GPUs may live in one process (any host thread).  Defined in
// murmur_api.cu; `slot` identifies the kernel.
enum SmemKernel { kSmemAttn = 0, kSmemStep, kSmemPrefill, kSmemPrefillUmma, kSmemIndexed, kSmemKernels };
cudaError_t opt_in_smem_once(int slot, const void* func, int smem);

// ---- host launchers (one per .cu) ------------------------------------------------------------
struct LaunchInfo {
  int launches;   // kernels launched
  int grid;       // CTAs of the main kernel
  int smem;       // dynamic smem of the main kernel
};

cudaError_t launch_init(const CacheView& c, cudaStream_t st, LaunchInfo* info);
cudaError_t launch_seq_begin(const CacheView& c, int seq, const SeqParams& sp, cudaStream_t st, LaunchInfo* info);
cudaError_t launch_seq_end(const CacheView& c, int seq, cudaStream_t st, LaunchInfo* info);
cudaError_t launch_append(const CacheView& c, const AppendList& list, int total_tokens, const void* k_new,
                          const void* v_new, int layer_begin, int layer_end, bool reserve, bool fuse_evict,
                          int sm_count, bool pdl, cudaStream_t st, LaunchInfo* info);
cudaError_t launch_evict(const CacheView& c, const SeqList& list, bool pdl, cudaStream_t st, LaunchInfo* info);
cudaError_t launch_attn_generic(const CacheView& c, const SeqList& list, int seq_base, int n_seqs_total,
                                const void* q, void* out, float* lse, int layer_begin, int layer_end,
                                float sm_scale, cudaStream_t st, LaunchInfo* info);
cudaError_t launch_attn_mma(const CacheView& c, const SeqList& list, int seq_base, int n_seqs_total, const void* q,
                            void* out, float* lse, int layer_begin, int layer_end, float sm_scale, int grid,
                            bool pdl, const SeqParams* window, cudaStream_t st, LaunchInfo* info);
// chain_expect >= 0: the previous launch on this handle's stream was a step launch; kCtrlStepDone reads that value
// once all of ITS keeper warps are done (see decode_attn_mma.cu, "chained steps").
cudaError_t launch_step_mma(const CacheView& c, const SeqList& list, const void* k_new, const void* v_new,
                            const void* q, void* out, float* lse, float sm_scale, int layer_begin, int layer_end,
                            bool write_only, int grid, bool pdl, long long chain_expect, cudaStream_t st, LaunchInfo* info);
cudaError_t launch_prefill_attn(const CacheView& c, int seq, int pos_begin, int n_tok, const void* q, void* out,
                                float* lse, int layer_begin, int layer_end, float sm_scale, cudaStream_t st,
                                LaunchInfo* info);
cudaError_t launch_prefill_attn_umma(const CacheView& c, int seq, int pos_begin, int n_tok, const void* q, void* out,
                                     float* lse, int layer_begin, int layer_end, float sm_scale, int sm_count,
                                     cudaStream_t st, LaunchInfo* info);
// member_mask (optional): uint8 [layers][n_seqs][n_kv][stride], set to 1 at the positions that belong to the mass
// set of ANY query head of the group; out may then be null.
cudaError_t launch_attn_profile(const CacheView& c, const SeqList& list, int seq_base, int n_seqs_total, const void* q,
                                const SeqParams* candidate, float frac, void* out, float* scratch, long long stride,
                                int layer_begin, int layer_end, float sm_scale, uint8_t* member_mask, cudaStream_t st,
                                LaunchInfo* info);
// The same launch with the library's built-in scratch array (attn_profile.cu); allocates nothing.
cudaError_t launch_attn_profile_noalloc(const CacheView& c, const SeqList& list, int n_seqs_total, const void* q,
                                        const SeqParams* candidate, float frac, void* out, long long stride,
                                        size_t scratch_bytes_needed, int layer_begin, int layer_end, float sm_scale,
                                        cudaStream_t st, LaunchInfo* info);
// Read-only validation of index sets (sizes, strict order, membership); *bad_dev must be 0 on entry.
cudaError_t launch_indexed_validate(const CacheView& c, const IdxView& ix, int seq, const int32_t* sel_pos,
                                    const int32_t* sel_cnt, int cap_sel, bool from_positional, int* bad_dev,
                                    cudaStream_t st, LaunchInfo* info);
cudaError_t launch_indexed_defrag(const CacheView& c, const IdxView& ix, int seq, const int32_t* sel_pos, const int32_t* sel_cnt,
                                  int cap_sel, bool from_positional, unsigned long long* moved_dev, cudaStream_t st,
                                  LaunchInfo* info);
cudaError_t launch_indexed_append(const CacheView& c, const IdxView& ix, const SeqList& list, const void* k_new,
                                  const void* v_new, cudaStream_t st, LaunchInfo* info);
cudaError_t launch_indexed_attn(const CacheView& c, const IdxView& ix, const SeqList& list, const void* q, void* out,
                                float* lse, float sm_scale, cudaStream_t st, LaunchInfo* info);
cudaError_t launch_indexed_attn_mma(const CacheView& c, const IdxView& ix, const SeqList& list, const void* q, void* out,
                                float* lse, float sm_scale, cudaStream_t st, LaunchInfo* info);
cudaError_t launch_indexed_gather(const CacheView& c, const IdxView& ix, int seq, void* k_out, void* v_out, int cap_out,
                                  cudaStream_t st, LaunchInfo* info);
cudaError_t launch_indexed_seq_end(const CacheView& c, int seq, cudaStream_t st, LaunchInfo* info);
cudaError_t launch_select_compact(const CacheView& c, int seq, const uint8_t* mask, long long mask_stride, int n_recent,
                                  int32_t* sel_pos, int32_t* sel_cnt, int cap_sel, cudaStream_t st, LaunchInfo* info);
cudaError_t launch_expand_retained(const CacheView& c, int seq, int32_t* pos_out_dev, int cap, cudaStream_t st,
                                   LaunchInfo* info);
cudaError_t launch_gather(const CacheView& c, int seq, const int32_t* positions_dev, int n, int layer_begin,
                          int layer_end, void* k_out, void* v_out, cudaStream_t st, LaunchInfo* info);

}  // namespace murmur
