/* murmur.h - C ABI of the B200-native MURMUR intra-chunk hot path.
 *
 * Paper: "MURMUR: An Efficient Inference System for Long-Form ASR" (arxiv/paper_2606_01483);
 * citations below are PAPER.md:<line> of the text mounted at /root/reference/PAPER.md.
 *
 * What the library computes, once per decode step and per layer:
 *   murmur_kv_append   - the newest token's K,V rows enter the KV cache C
 *   murmur_kv_evict    - the sliding-window eviction policy is applied: Alg. 1 on output
 *                        tokens, Eq. 2 / Alg. 2 on speech tokens
 *                        (PAPER.md:119-146), system prompts always kept;
 *                        dead pages are freed and the compacted page tables rebuilt
 *                        ("cache management")
 *   murmur_decode_attn - Eq. 1 softmax attention of one query token per
 *                        sequence over what remains, grouped-query, fp32 softmax
 *
 * Sequence layout: [prefix system prompt P][speech S][system prompt M][text t].
 * Positions are 0-based and absolute; t counts the output tokens in the cache INCLUDING the
 * newest one.  Retained ("attended") set at step t, region-relative indices r (speech), u (out):
 *     l(t)        = min(max(0, t - delay), max(0, S - w_speech))
 *     keep speech : r < n_sink_speech  or  l <= r < l + w_speech
 *     keep output : u < n_sink_out     or  u >= t - w_out
 *     keep prefix / mid always.
 * Tokens behind the trailing edge of their window (and not sinks) are dead for good; speech
 * tokens ahead of the window stay resident but are not attended.  See DESIGN.md "Readings".
 *
 * Memory model
 *   - The library never allocates device memory.  k_pool, v_pool and workspace are DEVICE
 *     buffers owned by the caller (e.g. torch tensors); they must outlive the handle and be
 *     256-byte aligned.  Sizes: murmur_pool_bytes() each for K and V, murmur_workspace_bytes().
 *   - Pool layout is PRIVATE (pre-swizzled for the attention kernel): read rows back only
 *     through murmur_kv_gather.
 *   - One physical page id addresses the same logical block in every layer and in K and V.
 *   - Arguments marked HOST are host pointers and are consumed before the call returns;
 *     arguments marked DEVICE are device pointers borrowed until the stream work completes.
 *   - `stream` is a cudaStream_t passed as void* (NULL = default stream).  All calls on one
 *     handle must be issued from one host thread at a time and on one stream (or on streams
 *     the caller orders).
 *
 * Errors: every call returns a murmur_status_t; nothing throws, aborts or prints.  Argument
 * and state errors (including page exhaustion, which the host-side mirror of the integer
 * state can always prove) are detected before any launch and leave all state unchanged.
 * The device additionally keeps an error word (murmur_get_last_error) as a cross-check.
 *
 * Order per decode step: append -> evict -> decode_attn (the query of output token t attends
 * a set containing token t itself: Alg. 1's K includes j).  evict twice at the
 * same t is a no-op.
 */
#ifndef MURMUR_H_
#define MURMUR_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(_WIN32)
#define MURMUR_API
#else
#define MURMUR_API __attribute__((visibility("default")))
#endif

typedef struct murmur_cache murmur_cache_t; /* opaque host object */

typedef enum {
  MURMUR_OK = 0,
  MURMUR_ERR_INVALID_ARG = 1, /* NULL pointer, out-of-range id, bad size, duplicate sequence in a call */
  MURMUR_ERR_STATE = 2,       /* sequence not active / already active / empty / max_blocks exceeded */
  MURMUR_ERR_OOM_PAGES = 3,   /* the call as a whole needs more pages than are free; nothing changed */
  MURMUR_ERR_CUDA = 4,        /* a CUDA runtime call failed */
  MURMUR_ERR_UNSUPPORTED = 5, /* geometry outside what the kernels are built for */
  MURMUR_ERR_SCRATCH_LIMIT = 6 /* murmur_attn_profile_noalloc only: the call needs more scratch than the library's
                                  built-in MURMUR_PROFILE_NOALLOC_MAX_BYTES; nothing was launched */
} murmur_status_t;

#define MURMUR_WINDOW_OFF 0x7fffffff /* window >= any length: that region is never evicted */
#define MURMUR_MAX_SEQS_PER_LAUNCH 128 /* larger calls are split internally, in order */

/* Geometry + caller-owned buffers.
 * Supported: head_dim == 128; n_q_heads % n_kv_heads == 0 with group size <= 8; page_size a power
 * of two in [1, 64] (the tensor-core attention path needs page_size >= 16; smaller pages use the
 * generic path); bf16 K/V/Q/O. */
typedef struct {
  int32_t n_layers, n_q_heads, n_kv_heads, head_dim; /* 28, 28, 4, 128 */
  int32_t page_size;                                 /* tokens per page */
  int32_t max_seqs;                                  /* sequence ids are 0 .. max_seqs-1 */
  int32_t max_blocks_per_seq;                        /* logical blocks (pages) a sequence may ever span */
  int64_t n_pages;                                   /* physical pages in each pool */
  void* k_pool;                                      /* DEVICE, murmur_pool_bytes() bytes */
  void* v_pool;                                      /* DEVICE, murmur_pool_bytes() bytes */
  void* workspace;                                   /* DEVICE, >= murmur_workspace_bytes() bytes */
  size_t workspace_bytes;
} murmur_cache_desc_t;

/* Per-sequence policy (paper names): w of Alg. 2, d of Alg. 2, n_sink of Eq. 2, w of Alg. 1,
 * n_sink of Alg. 1.  All >= 0.  MURMUR_WINDOW_OFF for a window disables that eviction. */
typedef struct {
  int32_t w_speech, delay, n_sink_speech, w_out, n_sink_out;
} murmur_policy_t;

/* Counters kept by the host object (what was launched through this handle). */
typedef struct {
  int64_t kernel_launches; /* CUDA kernels launched by this handle since creation / last reset */
  int64_t append_calls, evict_calls, attn_calls;
  int64_t free_pages;      /* host mirror of the free-stack height */
  int32_t attn_grid;       /* CTAs of the last attention launch */
  int32_t attn_smem_bytes; /* dynamic shared memory of the last attention launch */
  int32_t attn_variant;    /* variant used by the last attention launch (MURMUR_ATTN_*) */
  int32_t sm_count;
  int64_t host_zero_copy_steps; /* murmur_decode_step_host calls that ran on page-locked host buffers in place */
} murmur_stats_t;

/* Options for murmur_set_option. */
#define MURMUR_OPT_ATTN_VARIANT 1 /* value: MURMUR_ATTN_AUTO / _GENERIC / _MMA */
#define MURMUR_OPT_ATTN_GRID 2    /* value: CTAs for the persistent attention kernel; 0 = one per SM */
#define MURMUR_OPT_PDL 3          /* value: 1 (default) = kernels of a step are launched with programmatic
                                     dependent launch (each waits on-device for its predecessor), 0 = plain */
#define MURMUR_OPT_FUSE_STEP 4    /* murmur_decode_step as: 2 (default) = ONE launch (the attention CTAs derive the
                                     post-append state themselves, keeper warps scatter the rows, commit and evict;
                                     needs the tensor-core attention variant and <= 64 sequences in the call,
                                     else falls back to 1);
                                     1 = two launches (append with the eviction fused in, then attention);
                                     0 = three launches (append, evict, attention) */
#define MURMUR_OPT_HOST_ZERO_COPY 6 /* value: 1 (default) = murmur_decode_step_host works on page-locked host buffers
                                      in place (zero-copy); 0 = always stage through device buffers */
#define MURMUR_OPT_L2_KEEP_PCT 7   /* value: 0 (default) .. 100: percentage of the K/V rows a decode-attention launch reads
                                      with L2::evict_last instead of L2::evict_first - the retained set of step t+1 is that
                                      of step t shifted by one token, so whatever part of it fits the L2 can be served from
                                      there on the next step; -1 = automatic (half an L2 when the retained rows of the
                                      sequences in the call are at most 1.3 L2 sizes, else none).  Opt-in because pinned
                                      lines are never demoted and take L2 from whatever else runs between two attention
                                      calls; results do not depend on it */
#define MURMUR_OPT_PREFILL_VARIANT 5 /* value: MURMUR_PREFILL_AUTO / _MMA_SYNC / _UMMA */
#define MURMUR_PREFILL_AUTO 0     /* = MURMUR_PREFILL_UMMA */
#define MURMUR_PREFILL_MMA_SYNC 1 /* warp-level mma.sync kernel (the round-1 path, kept as a cross-check) */
#define MURMUR_PREFILL_UMMA 2     /* tcgen05.mma, accumulators in tensor memory, TMA-fed operands */
#define MURMUR_ATTN_AUTO 0    /* tensor-core split-K kernel when page_size >= 16, else generic */
#define MURMUR_ATTN_GENERIC 1 /* one CTA per (layer, sequence, KV head), FFMA, no smem staging */
#define MURMUR_ATTN_MMA 2     /* persistent split-K kernel: bulk-copy staging + mma.sync bf16 */

/* ---- sizing ------------------------------------------------------------------------------ */
/* Bytes of ONE pool (K or V): n_layers * n_pages * n_kv_heads * page_size * head_dim * 2. */
MURMUR_API size_t murmur_pool_bytes(const murmur_cache_desc_t* desc);
/* Bytes of workspace the handle needs (page tables, free stack, split-K partials, staging).
 * Returns 0 if desc is NULL or unsupported. */
MURMUR_API size_t murmur_workspace_bytes(const murmur_cache_desc_t* desc);

/* ---- lifecycle --------------------------------------------------------------------------- */
/* Creates the handle and initialises the workspace on `stream` (free stack = all pages, pops
 * return page 0,1,2,...).  Pool contents are not touched.  *out is set only on MURMUR_OK. */
MURMUR_API murmur_status_t murmur_cache_create(const murmur_cache_desc_t* desc, murmur_cache_t** out, void* stream);
/* Frees the host object only (device buffers belong to the caller). NULL is a no-op. */
MURMUR_API murmur_status_t murmur_cache_destroy(murmur_cache_t* cache);

/* Declares sequence `seq` with its region sizes and policy; it starts empty.  The first
 * n_prefix + n_speech + n_mid tokens appended are the prefill, later ones are output tokens. */
MURMUR_API murmur_status_t murmur_seq_begin(murmur_cache_t* cache, int32_t seq, int32_t n_prefix, int32_t n_speech,
                                            int32_t n_mid, const murmur_policy_t* policy, void* stream);
/* Ends the sequence; its live pages are pushed on the free stack in ascending block order. */
MURMUR_API murmur_status_t murmur_seq_end(murmur_cache_t* cache, int32_t seq, void* stream);

/* ---- the hot path ------------------------------------------------------------------------ */
/* Appends n_tokens[i] tokens to sequence seq_ids[i].
 *   seq_ids, n_tokens : HOST int32[n_seqs]; ids distinct and active; n_tokens[i] >= 0.
 *   k_new, v_new      : DEVICE bf16 [layer_end-layer_begin][sum n_tokens][n_kv_heads][head_dim],
 *                       tokens of a sequence contiguous, sequences in call order.
 *   layer_begin == 0 reserves the slots (allocating pages in call order, new blocks ascending;
 *   all-or-nothing) and advances the sequence lengths; a call with layer_begin > 0 only writes
 *   rows for the LAST n_tokens[i] reserved positions (engines that produce layer l's K/V at
 *   layer l call it once per layer range).  Bulk prefill and 1-token decode use the same call. */
MURMUR_API murmur_status_t murmur_kv_append(murmur_cache_t* cache, const int32_t* seq_ids, const int32_t* n_tokens,
                                            int32_t n_seqs, const void* k_new, const void* v_new,
                                            int32_t layer_begin, int32_t layer_end, void* stream);

/* Applies each sequence's policy at its current t: frees blocks whose every
 * position is dead (sequences in call order, blocks ascending), rebuilds the compacted live-page
 * list, the run descriptors (maximal intervals of the retained set) and the attention work
 * list.  No K/V bytes move.  seq_ids: HOST int32[n_seqs], distinct, active. */
MURMUR_API murmur_status_t murmur_kv_evict(murmur_cache_t* cache, const int32_t* seq_ids, int32_t n_seqs, void* stream);

/* Eq. 1: out[l][i][h] = sum_x alpha_x v_x over the retained set of seq_ids[i]
 * as of its last murmur_kv_evict, alpha = softmax(q . k_x * sm_scale), KV head of query head h
 * is h / (n_q_heads / n_kv_heads).
 *   q, out : DEVICE bf16 [layer_end-layer_begin][n_seqs][n_q_heads][head_dim]
 *   lse    : DEVICE fp32 [layer_end-layer_begin][n_seqs][n_q_heads] natural-log-sum-exp of the
 *            scaled scores, or NULL
 * Every listed sequence must have a non-empty retained set and have been evicted since its last
 * append (else MURMUR_ERR_STATE). */
MURMUR_API murmur_status_t murmur_decode_attn(murmur_cache_t* cache, const int32_t* seq_ids, int32_t n_seqs,
                                              const void* q, void* out, float* lse, int32_t layer_begin,
                                              int32_t layer_end, float sm_scale, void* stream);

/* Per-layer windows (sparsity differs by layer; "particularly in deeper layers"): the same
 * as murmur_decode_attn, but the attended set of every listed sequence is the A(t) of `window` (HOST)
 * instead of its own policy's - call it once per group of layers that share a window.  What is RESIDENT
 * is still decided by each sequence's own policy (murmur_kv_evict), which therefore has to be the
 * loosest one: `window` may not exceed it in any field (else MURMUR_ERR_INVALID_ARG), so that A_window(t)
 * never touches an evicted position.  Tensor-core variant only (page_size >= 16). */
MURMUR_API murmur_status_t murmur_decode_attn_windowed(murmur_cache_t* cache, const int32_t* seq_ids, int32_t n_seqs,
                                                       const void* q, void* out, float* lse, int32_t layer_begin,
                                                       int32_t layer_end, float sm_scale,
                                                       const murmur_policy_t* window, void* stream);

/* One whole decode step from DEVICE buffers: append one token to every listed sequence (all
 * layers) -> evict -> decode_attn, enqueued by ONE host call as ONE launch by default (see
 * MURMUR_OPT_FUSE_STEP; the result is identical for every setting) (PAPER.md:112-116, 136-146, 101-104:
 * the per-step loop body of Alg. 1 / Alg. 2 followed by Eq. 1).
 *   k_new, v_new : DEVICE bf16 [n_layers][n_seqs][n_kv_heads][head_dim]
 *   q, out       : DEVICE bf16 [n_layers][n_seqs][n_q_heads][head_dim];  lse as above or NULL
 * n_seqs <= MURMUR_MAX_SEQS_PER_LAUNCH.  Validated as a whole before anything is enqueued. */
MURMUR_API murmur_status_t murmur_decode_step(murmur_cache_t* cache, const int32_t* seq_ids, int32_t n_seqs,
                                              const void* k_new, const void* v_new, const void* q, void* out,
                                              float* lse, float sm_scale, void* stream);

/* The decode step of an engine that produces layer l's K/V only when layer l runs (cache
 * management must not eat the gain): the same step restricted to the layers [layer_begin, layer_end), ONE launch
 * per call.  The call with layer_begin == 0 OPENS the step - it reserves the new token's slot in every listed
 * sequence, advances the lengths and runs the eviction - and must come first; calls with layer_begin > 0 only
 * write their layers' rows and attend (MURMUR_ERR_STATE unless the step is open for every listed sequence;
 * rows of a token the open step's eviction already freed are dropped).  Layer ranges may be issued in any
 * order and size after the opening one, each layer ONCE: the step closes when every layer has been issued, and a
 * range that touches a layer already issued in this step, or comes after a murmur_kv_append / murmur_kv_evict of
 * the sequence, is MURMUR_ERR_STATE.  murmur_decode_step == one call with [0, n_layers).
 *   k_new, v_new : DEVICE bf16 [layer_end-layer_begin][n_seqs][n_kv_heads][head_dim]
 *   q, out       : DEVICE bf16 [layer_end-layer_begin][n_seqs][n_q_heads][head_dim];  lse likewise or NULL */
MURMUR_API murmur_status_t murmur_decode_step_layers(murmur_cache_t* cache, const int32_t* seq_ids, int32_t n_seqs,
                                                     const void* k_new, const void* v_new, const void* q, void* out,
                                                     float* lse, int32_t layer_begin, int32_t layer_end,
                                                     float sm_scale, void* stream);

/* The whole step issued from C as ceil(n_layers / layers_per_launch) launches of murmur_decode_step_layers, in
 * layer order (buffers as for murmur_decode_step).  layers_per_launch = 1 is the launch pattern of a
 * layer-by-layer engine (what bench.py reports as per_layer_mode_us); the host-buffer entry uses larger chunks
 * to overlap its copies with the kernels.  layers_per_launch >= n_layers == murmur_decode_step. */
MURMUR_API murmur_status_t murmur_decode_step_chunked(murmur_cache_t* cache, const int32_t* seq_ids, int32_t n_seqs,
                                                      const void* k_new, const void* v_new, const void* q, void* out,
                                                      float* lse, int32_t layers_per_launch, float sm_scale,
                                                      void* stream);

/* One whole decode step from HOST buffers (the end-to-end entry): k_new, v_new, q in, out back (HOST bf16, layouts
 * as for murmur_decode_step with all layers), all on `stream`; returns after enqueueing (synchronise the stream
 * before reading out_host).  n_seqs <= MURMUR_MAX_SEQS_PER_LAUNCH.
 *   Page-locked buffers (cudaHostAlloc, cudaHostRegister, torch pin_memory; all four, 16-byte aligned): ZERO-COPY -
 *   the one-launch step kernel reads q / k_new / v_new from the host buffers and stores out to the host buffer
 *   itself, through their device-mapped addresses; the data crosses PCIe inside the kernel, overlapped with the
 *   K/V stream from HBM, and there is no staging copy.  MURMUR_OPT_HOST_ZERO_COPY = 0 turns this off.
 *   Pageable buffers: staged - cudaMemcpyAsync to device staging (one copy if k_new, v_new, q are packed back to
 *   back), the step, cudaMemcpyAsync of out back. */
MURMUR_API murmur_status_t murmur_decode_step_host(murmur_cache_t* cache, const int32_t* seq_ids, int32_t n_seqs,
                                                   const void* k_new_host, const void* v_new_host,
                                                   const void* q_host, void* out_host, float sm_scale, void* stream);

/* CUDA graphs.  Every state transition of a step runs on the device, so a captured murmur_decode_step (or the
 * murmur_decode_step_layers calls of one step) can be REPLAYED: capture the call(s) once with fixed k_new / v_new / q /
 * out buffers (after at least one un-captured step, so that one-time kernel attributes are set), refill the buffers and
 * replay once per decode step.  Replays bypass the host-side validation (the kernels keep the device error word: page
 * exhaustion or max_blocks_per_seq raise it and the step does nothing) and the host mirror of lengths and free pages.
 * Call murmur_mirror_sync (synchronises `stream`) before the next non-replayed call on the handle; it re-reads lengths
 * and the free-stack height from the device.  This is enforced: once a call has been recorded into a graph, every
 * state-dependent call made outside a capture (sequence begin / end, append, evict, attention, step, prefill, the
 * indexed calls) returns MURMUR_ERR_STATE until murmur_mirror_sync has run; introspection, options and statistics
 * stay available.  Sequences may not begin or end inside a replayed stretch. */
MURMUR_API murmur_status_t murmur_mirror_sync(murmur_cache_t* cache, void* stream);

/* ---- chunking (host only) ------------------------------------------------------------------ */
/* Greedy merge of VAD speech segments into chunks of span <= max_len seconds (c = 300 s).
 *   seg_start, seg_end : HOST float[n_segments], seconds, sorted and non-overlapping
 *   chunk_first_seg    : HOST int32[cap] out: index of the first segment of each chunk (chunk j covers
 *                        segments chunk_first_seg[j] .. chunk_first_seg[j+1]-1); may be NULL with cap 0
 *   *n_chunks_out      : number of chunks (set even when cap is too small -> MURMUR_ERR_INVALID_ARG)
 * A segment longer than max_len is a chunk by itself.  No GPU work, no handle. */
MURMUR_API murmur_status_t murmur_chunk_plan(const float* seg_start, const float* seg_end, int32_t n_segments,
                                             float max_len, int32_t* chunk_first_seg, int32_t cap,
                                             int32_t* n_chunks_out);

/* Batch formation ("Chunks are submitted as a batch to an inference engine"; "a batch size of
 * 16 chunks" and the maximum-new-tokens rule).  For the chunks murmur_chunk_plan produced (same segment arrays,
 * chunk_first_seg HOST int32[n_chunks], n_chunks <= n_segments), entry j describes chunk j:
 *   batch, slot  chunks stay in time order and fill consecutive batches of batch_size: j / batch_size, j % batch_size
 *                (slot = the sequence id to use in that batch's handle)
 *   n_speech     S = ceil(tokens_per_s * d), d = the chunk's span in seconds (first segment's start to last one's end);
 *                BASELINE.json's rate is 7.5 (300 s -> 2250 tokens)
 *   max_new      T = floor(max_new_nominal * d / d_nominal) for d < d_nominal, else max_new_nominal; at least 1
 *                (the paper: 32768 and 3600 s)
 *   max_blocks   ceil((n_prefix + S + n_mid + T) / page_size): what murmur_cache_desc_t.max_blocks_per_seq must cover
 * so that murmur_seq_begin(cache_of(batch), slot, n_prefix, n_speech, n_mid, policy) can follow directly.
 *   entries        : HOST murmur_batch_entry_t[n_chunks] out;  *n_batches_out = ceil(n_chunks / batch_size)
 * Decisions are taken in IEEE double.  MURMUR_ERR_INVALID_ARG on NULL / non-positive parameters, a chunk table that is
 * not strictly ascending from 0, or a geometry that does not fit int32.  No GPU work, no handle. */
typedef struct {
  int32_t chunk, batch, slot, n_speech, max_new, max_blocks;
} murmur_batch_entry_t;
MURMUR_API murmur_status_t murmur_batch_plan(const float* seg_start, const float* seg_end, int32_t n_segments,
                                             const int32_t* chunk_first_seg, int32_t n_chunks, int32_t batch_size,
                                             double tokens_per_s, int32_t max_new_nominal, double d_nominal,
                                             int32_t n_prefix, int32_t n_mid, int32_t page_size,
                                             murmur_batch_entry_t* entries, int32_t* n_batches_out);

/* ---- prefill ------------------------------------------------------------------------------- */
/* Causal self-attention of prefill tokens: for the positions x in
 * [pos_begin, pos_end) of `seq`, out[l][x - pos_begin][h] = Eq. 1 of query q_x over
 * the cache positions y <= x.  The K/V of positions [0, pos_end) must already be appended for the
 * given layers and none of them evicted (MURMUR_ERR_STATE otherwise) - call it after the bulk
 * murmur_kv_append of the chunk and before the first murmur_kv_evict.
 *   q, out : DEVICE bf16 [layer_end-layer_begin][pos_end-pos_begin][n_q_heads][head_dim]
 *   lse    : DEVICE fp32 [layer_end-layer_begin][pos_end-pos_begin][n_q_heads] or NULL
 * page_size >= 16; q and out 16-byte aligned.  Runs on the 5th-generation tensor cores (tcgen05.mma, accumulators in
 * tensor memory, operands staged by TMA straight from the paged pools); MURMUR_OPT_PREFILL_VARIANT selects the
 * warp-level mma.sync kernel instead. */
MURMUR_API murmur_status_t murmur_prefill_attn(murmur_cache_t* cache, int32_t seq, int32_t pos_begin, int32_t pos_end,
                                               const void* q, void* out, float* lse, int32_t layer_begin,
                                               int32_t layer_end, float sm_scale, void* stream);

/* ---- analysis: attention-sparsity profile (Fig. 5 at PAPER.md:85) ----------------- */
/* Per (layer, sequence, query head), over the RESIDENT positions of the cache (everything not dead;
 * run the cache with MURMUR_WINDOW_OFF to profile full attention):
 *   n_*        tokens per region: prompt = both system prompts, speech, text = output tokens
 *   k_mass     size of the FEWEST-token set whose Eq. 1 weights sum to >= mass_frac of the total
 *              (weights descending, ties by ascending position); k_prompt/k_speech/k_text = its
 *              members per region ("kept" of Fig. 5; "evictable" = n_* - k_*)
 *   mass_*     attention mass per region;  coverage = mass inside the retained set A(t) of the
 *              candidate policy (what a window policy would preserve at this step) */
typedef struct {
  int32_t n_resident, n_prompt, n_speech, n_text;
  int32_t k_mass, k_prompt, k_speech, k_text;
  float coverage, mass_prompt, mass_speech, mass_text;
} murmur_profile_t;

/* Bytes of DEVICE scratch murmur_attn_profile needs for these sequences and layers (0 on bad arguments). */
MURMUR_API size_t murmur_profile_scratch_bytes(murmur_cache_t* cache, const int32_t* seq_ids, int32_t n_seqs,
                                               int32_t layer_begin, int32_t layer_end);
/* q        : DEVICE bf16 [layer_end-layer_begin][n_seqs][n_q_heads][head_dim] (the step's queries)
 * candidate: HOST policy whose A(t) `coverage` is measured against, or NULL = each sequence's own
 * mass_frac: in (0, 1], the paper uses 0.99
 * out      : DEVICE murmur_profile_t [layer_end-layer_begin][n_seqs][n_q_heads]
 * scratch  : DEVICE, >= murmur_profile_scratch_bytes(); n_seqs <= MURMUR_MAX_SEQS_PER_LAUNCH.
 * Reads the cache only (any time after an append; no evict needed); softmax in fp32, sums in fp64. */
MURMUR_API murmur_status_t murmur_attn_profile(murmur_cache_t* cache, const int32_t* seq_ids, int32_t n_seqs,
                                               const void* q, const murmur_policy_t* candidate, float mass_frac,
                                               void* out, void* scratch, size_t scratch_bytes, int32_t layer_begin,
                                               int32_t layer_end, float sm_scale, void* stream);

/* murmur_attn_profile for callers that have no way to get a scratch buffer.
 *
 * Who that is: murmur_attn_profile wants murmur_profile_scratch_bytes() of device memory from the caller, and the
 * amount depends on how long the sequences are at the moment of the call.  Some callers cannot produce that:
 *   - a monitoring hook inside a serving engine that handed ALL device memory to its KV pool and activation arena
 *     at start-up and forbids (or simply fails) any later cudaMalloc;
 *   - code running on a latency-critical decode loop, where cudaMalloc / cudaFree would stall the whole GPU (both
 *     synchronise the device) for a profile that is sampled once in a while;
 *   - plug-in code called from someone else's runtime (a callback, a foreign-language binding) that is given the
 *     step's tensors but no handle to that runtime's allocator.
 * For them the library carries its own scratch: a fixed array of MURMUR_PROFILE_NOALLOC_MAX_BYTES in the library's
 * device image.  Every GPU that loads the library holds those bytes from load until process exit, used or not -
 * that is why the limit is modest.  The call allocates nothing: no cudaMalloc, no cudaFree, no library routine that
 * allocates; q and out are still the caller's.
 *
 * Arguments, result and errors are those of murmur_attn_profile (Fig. 5 at PAPER.md:85), without
 * scratch / scratch_bytes.  In addition:
 *   - MURMUR_ERR_SCRATCH_LIMIT when murmur_profile_scratch_bytes(cache, seq_ids, n_seqs, layer_begin, layer_end)
 *     exceeds MURMUR_PROFILE_NOALLOC_MAX_BYTES; nothing is launched.  The need is (layers in the call) x n_seqs x
 *     n_q_heads x (longest listed sequence, rounded up to 32) x 4 bytes: 8 MiB is e.g. one layer of 16 sequences of
 *     4 600 tokens at 28 heads, or one 2 314-token sequence over all 28 layers.  Split larger jobs by layer range.
 *   - The FIRST call on each GPU also looks up where the array lives on that GPU (with that GPU current, as for
 *     every call on the handle).  Make that first call during set-up, before any stream capture is begun.
 *   - The array is shared by everything in the process that uses this GPU and keeps the previous call's contents.
 *     That is harmless for a single call (the kernel writes every element it later reads; nothing has to start at
 *     zero), but two calls that overlap on the GPU - different streams, handles or threads - overwrite each other's
 *     rows and both results are garbage.  Issue them on one stream or order them with events. */
#define MURMUR_PROFILE_NOALLOC_MAX_BYTES (8u << 20)
MURMUR_API murmur_status_t murmur_attn_profile_noalloc(murmur_cache_t* cache, const int32_t* seq_ids, int32_t n_seqs,
                                                       const void* q, const murmur_policy_t* candidate,
                                                       float mass_frac, void* out, int32_t layer_begin,
                                                       int32_t layer_end, float sm_scale, void* stream);

/* ---- general index-set eviction: "indexed mode" --------------------------------------------
 * "The evictable tokens are not contiguous and cannot be captured by a simple positional policy. This motivates
 * future work on ... query-aware ... eviction policies"; the sparsity is per layer and head
 * (PAPER.md:29, 77, 99).  These calls are the cache side of such policies (definitions: DESIGN.md "f3" - a
 * convention of this build, the paper defines none):
 *   index set     per (layer l, KV head h), an ascending list of ORIGINAL absolute positions to keep;
 *   indexed mode  the sequence's rows are stored densely per slab (l, h): slot s holds the row of the s-th smallest
 *                 retained position (dense, stable: order preserved); slabs have different lengths;
 *   pages         a page id still addresses one logical block in every layer and head, so the sequence keeps blocks
 *                 0 .. ceil(longest slab / page_size) - 1; surplus pages go back on the free stack, ascending.
 * A sequence enters indexed mode with its first murmur_kv_evict_indexed and stays there; the positional calls
 * (murmur_kv_append / _evict / _decode_attn / _decode_step / _prefill_attn / _kv_gather) then return MURMUR_ERR_STATE
 * for it and the *_indexed calls take over.  murmur_seq_end works in both modes. */
/* Bytes of the DEVICE buffer murmur_indexed_enable needs (slab lengths + position tables); 0 if unsupported. */
MURMUR_API size_t murmur_indexed_bytes(const murmur_cache_desc_t* desc);
/* Hands the handle a caller-owned DEVICE buffer (256-byte aligned, >= murmur_indexed_bytes()) for the indexed-mode
 * tables; it must outlive the handle.  MURMUR_ERR_STATE while any sequence is in indexed mode. */
MURMUR_API murmur_status_t murmur_indexed_enable(murmur_cache_t* cache, void* buffer, size_t bytes, void* stream);
/* Query-aware index sets from the quantity the paper measures (Fig. 5 at PAPER.md:85): for every
 * (layer, KV head), the union over the query heads of the group of each head's fewest-token set holding >= mass_frac
 * of its Eq. 1 mass over the resident positions (as murmur_attn_profile finds it), plus both system prompts
 * (never evicted) and the n_recent newest positions.  `seq` must be positional (not yet indexed).
 *   q        : DEVICE bf16 [n_layers][n_q_heads][head_dim] (the step's queries of this sequence)
 *   sel_pos  : DEVICE int32 [n_layers][n_kv_heads][cap] out, ascending;  sel_cnt: DEVICE int32 [n_layers][n_kv_heads] out
 *   scratch  : DEVICE, >= murmur_select_scratch_bytes()
 * A set larger than cap raises the device error word (its count is still written). */
MURMUR_API size_t murmur_select_scratch_bytes(murmur_cache_t* cache, int32_t seq);
MURMUR_API murmur_status_t murmur_select_mass_sets(murmur_cache_t* cache, int32_t seq, const void* q, float mass_frac,
                                                   int32_t n_recent, int32_t* sel_pos, int32_t* sel_cnt, int32_t cap,
                                                   void* scratch, size_t scratch_bytes, float sm_scale, void* stream);
/* Applies index sets (layouts as above, DEVICE, each set strictly ascending, a subset of what its slab holds, >= 1
 * element): afterwards slot s of slab (l, h) holds the row of position sel_pos[l][h][s] and everything else is gone.
 * The compaction is in place (rows only move towards lower addresses); *bytes_moved_out (HOST, may be NULL) = bytes of
 * K/V rows that changed address - the cost of cache management made countable.  A positional
 * sequence must have been evicted since its last append (its live page list is the source).  SYNCHRONISES the stream
 * (the set sizes are read back for the page accounting).  The sets are validated on the device before any row moves:
 * a set that is empty, larger than cap, not strictly ascending, or names a position its slab does not hold returns
 * MURMUR_ERR_INVALID_ARG with the sequence, its rows, its pages and its mode unchanged. */
MURMUR_API murmur_status_t murmur_kv_evict_indexed(murmur_cache_t* cache, int32_t seq, const int32_t* sel_pos,
                                                   const int32_t* sel_cnt, int32_t cap, int64_t* bytes_moved_out,
                                                   void* stream);
/* Appends ONE token to every slab of every listed (indexed-mode) sequence; its original position is the sequence's
 * running token count.  A page is popped when a sequence's longest slab starts a new block (call order; all-or-nothing).
 *   k_new, v_new : DEVICE bf16 [n_layers][n_seqs][n_kv_heads][head_dim] */
MURMUR_API murmur_status_t murmur_kv_append_indexed(murmur_cache_t* cache, const int32_t* seq_ids, int32_t n_seqs,
                                                    const void* k_new, const void* v_new, void* stream);
/* Eq. 1 of every query head hq over the rows of slab (l, hq / group), all layers.
 *   q, out : DEVICE bf16 [n_layers][n_seqs][n_q_heads][head_dim];  lse: DEVICE fp32 [n_layers][n_seqs][n_q_heads] or NULL
 * page_size >= 16: the streaming tensor-core kernel (one CTA per slab: bulk-copy ring, mma.sync, fragment-layout
 * merge); smaller pages: FFMA straight from the pool. */
MURMUR_API murmur_status_t murmur_decode_attn_indexed(murmur_cache_t* cache, const int32_t* seq_ids, int32_t n_seqs,
                                                      const void* q, void* out, float* lse, float sm_scale, void* stream);
/* Introspection (synchronise): the original positions held by slab (layer, kv_head), by slot; and the rows of every
 * slab by slot, k_out / v_out DEVICE bf16 [n_layers][n_kv_heads][cap_rows][head_dim] (zero beyond a slab's length). */
MURMUR_API murmur_status_t murmur_kv_get_indexed(murmur_cache_t* cache, int32_t seq, int32_t layer, int32_t kv_head,
                                                 int32_t* pos_out, int32_t cap, int32_t* n_out, void* stream);
MURMUR_API murmur_status_t murmur_kv_gather_indexed(murmur_cache_t* cache, int32_t seq, void* k_out, void* v_out,
                                                    int32_t cap_rows, void* stream);

/* ---- introspection (tests; each call synchronises the stream it is given) ------------------ */
/* state_out[0..5] = length, t, n_live_blocks, n_runs, n_attn_tiles, n_retained (device values). */
MURMUR_API murmur_status_t murmur_seq_get_state(murmur_cache_t* cache, int32_t seq, int32_t* state_out, void* stream);
/* Sorted absolute positions of the retained set (expanded on the device from the run descriptors). */
MURMUR_API murmur_status_t murmur_kv_get_retained(murmur_cache_t* cache, int32_t seq, int32_t* pos_out, int32_t cap,
                                                  int32_t* n_out, void* stream);
/* Compacted page table: physical ids and logical block numbers of the live blocks, ascending. */
MURMUR_API murmur_status_t murmur_kv_get_page_list(murmur_cache_t* cache, int32_t seq, int32_t* pages_out,
                                                   int32_t* blocks_out, int32_t cap, int32_t* n_out, void* stream);
/* Run descriptors: runs_out[3*k+0..2] = first_pos, n_tok, index of the run's first block in the page list. */
MURMUR_API murmur_status_t murmur_kv_get_runs(murmur_cache_t* cache, int32_t seq, int32_t* runs_out, int32_t cap_runs,
                                              int32_t* n_out, void* stream);
/* Free stack, bottom to top (the next pop returns the last element). */
MURMUR_API murmur_status_t murmur_kv_get_free_stack(murmur_cache_t* cache, int32_t* pages_out, int64_t cap,
                                                    int64_t* n_out, void* stream);
/* Gathers the K and V rows of n positions (HOST int32[n], all resident) of one sequence into
 * k_out, v_out: DEVICE bf16 [layer_end-layer_begin][n][n_kv_heads][head_dim], natural order. */
MURMUR_API murmur_status_t murmur_kv_gather(murmur_cache_t* cache, int32_t seq, const int32_t* positions, int32_t n,
                                            int32_t layer_begin, int32_t layer_end, void* k_out, void* v_out,
                                            void* stream);
/* Device error word: 0 or the first MURMUR_ERR_* a kernel detected since creation. */
MURMUR_API murmur_status_t murmur_get_last_error(murmur_cache_t* cache, int32_t* device_err_out, void* stream);

#ifdef MURMUR_TRACE
/* Profiling builds only (library compiled with -DMURMUR_TRACE: `python -m paper_2606_01483_b200.build --trace`);
 * the production kernels carry no time stamps and the production library does not export these. */
#define MURMUR_TRACE_API MURMUR_API
/* Per-CTA trace of the LAST tensor-core attention launch: out is HOST uint64[n][8] = {globaltimer ns when
 * the CTA started its work (after the chain / dependency wait), at CTA end, SM id, tiles processed, ns at kernel
 * entry, set-up done, keeper past its dependency wait, keeper done}; *n_out = CTAs of that launch (0 if the
 * last launch was the generic variant). */
MURMUR_TRACE_API murmur_status_t murmur_debug_attn_timeline(murmur_cache_t* cache, uint64_t* out, int32_t cap_ctas,
                                                            int32_t* n_out, void* stream);
/* globaltimer stamps (ns) of the LAST step prologue, HOST uint64[16]:
 * [0] append kernel start (CTA 0, after its dependency wait)  [1] last append CTA through the ticket
 * [2] integer state committed  [3] eviction body start  [4] eviction body end;  the last CTA's own
 * phases: [5] after its dependency wait [6] old state loaded [7] prefix sums done [8] row loads
 * issued [9] eviction tasks done [10] page ids consumed [11] its block index; rest unused. */
MURMUR_TRACE_API murmur_status_t murmur_debug_step_trace(murmur_cache_t* cache, uint64_t* out16, void* stream);
#endif

/* ---- options / stats --------------------------------------------------------------------- */
MURMUR_API murmur_status_t murmur_set_option(murmur_cache_t* cache, int32_t option, int32_t value);
MURMUR_API murmur_status_t murmur_get_stats(murmur_cache_t* cache, murmur_stats_t* out);
MURMUR_API murmur_status_t murmur_reset_stats(murmur_cache_t* cache);
MURMUR_API const char* murmur_status_str(murmur_status_t s);
/* Text of the CUDA error behind the last MURMUR_ERR_CUDA returned through this handle. */
MURMUR_API const char* murmur_last_cuda_error(murmur_cache_t* cache);
MURMUR_API const char* murmur_version(void);

#ifdef __cplusplus
}
#endif
#endif /* MURMUR_H_ */
