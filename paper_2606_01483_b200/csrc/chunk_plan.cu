// murmur_chunk_plan: greedy merge of VAD speech segments into chunks of at most max_len seconds.
//
// "Segments are greedily merged to construct chunks {C_1..C_m} where each chunk
// satisfies |C_i| <= c = 300 s"; the chunks are then submitted as one batch (the sequences of a
// murmur_decode_step call).  Host logic only - it runs once per recording, before any GPU work.
// Readings (G23): |C| is the span from the start of the chunk's first segment to the end
// of its last one (silences inside count: that audio is fed to the model); a single segment longer
// than max_len cannot be merged with anything and forms a chunk of its own.
#include <math.h>

#include "../../include/murmur.h"

extern "C" murmur_status_t murmur_chunk_plan(const float* seg_start, const float* seg_end, int32_t n_segments,
                                             float max_len, int32_t* chunk_first_seg, int32_t cap,
                                             int32_t* n_chunks_out) {
  if (n_segments < 0 || !n_chunks_out || !(max_len > 0.f)) return MURMUR_ERR_INVALID_ARG;
  if (n_segments > 0 && (!seg_start || !seg_end)) return MURMUR_ERR_INVALID_ARG;
  for (int32_t i = 0; i < n_segments; ++i) {
    if (!(seg_end[i] >= seg_start[i])) return MURMUR_ERR_INVALID_ARG;
    if (i > 0 && !(seg_start[i] >= seg_end[i - 1])) return MURMUR_ERR_INVALID_ARG;  // sorted, non-overlapping
  }
  int32_t n = 0;
  float chunk_start = 0.f;
  for (int32_t i = 0; i < n_segments; ++i) {
    if (n == 0 || seg_end[i] - chunk_start > max_len) {  // does not fit the open chunk: start a new one
      if (n < cap && chunk_first_seg) chunk_first_seg[n] = i;
      ++n;
      chunk_start = seg_start[i];
    }
  }
  *n_chunks_out = n;
  return (n > cap) ? MURMUR_ERR_INVALID_ARG : MURMUR_OK;
}

// murmur_batch_plan: the chunks of a recording -> batches of sequence slots with the geometry murmur_seq_begin and
// the cache descriptor need.
//
// "Chunks are submitted as a batch to an inference engine"; "a batch size of 16 chunks",
// "The maximum number of new tokens is set to 32,768 for recordings within the model's nominal context length of 60
// minutes; for shorter recordings, it is scaled as |32,768 x d/d_nominal|".  Readings (G24-G26): chunks
// stay in time order and fill consecutive batches; a chunk's duration d is its span (G23); S = ceil(rate * d) speech
// tokens; T = floor(max_new_nominal * d / d_nominal) below the nominal duration, max_new_nominal from there on, never
// less than 1.  The decisions are taken in IEEE double on the float32 times, in the order written here.
extern "C" murmur_status_t murmur_batch_plan(const float* seg_start, const float* seg_end, int32_t n_segments,
                                             const int32_t* chunk_first_seg, int32_t n_chunks, int32_t batch_size,
                                             double tokens_per_s, int32_t max_new_nominal, double d_nominal,
                                             int32_t n_prefix, int32_t n_mid, int32_t page_size,
                                             murmur_batch_entry_t* entries, int32_t* n_batches_out) {
  if (!n_batches_out || n_segments < 0 || n_chunks < 0 || n_chunks > n_segments) return MURMUR_ERR_INVALID_ARG;
  if (batch_size < 1 || !(tokens_per_s > 0.0) || max_new_nominal < 1 || !(d_nominal > 0.0)) return MURMUR_ERR_INVALID_ARG;
  if (n_prefix < 0 || n_mid < 0 || page_size < 1) return MURMUR_ERR_INVALID_ARG;
  if (n_chunks > 0 && (!seg_start || !seg_end || !chunk_first_seg || !entries)) return MURMUR_ERR_INVALID_ARG;
  for (int32_t j = 0; j < n_chunks; ++j) {  // first segments strictly ascending, starting at 0
    const int32_t f = chunk_first_seg[j];
    if (f < 0 || f >= n_segments || (j == 0 ? f != 0 : f <= chunk_first_seg[j - 1])) return MURMUR_ERR_INVALID_ARG;
  }
  for (int32_t j = 0; j < n_chunks; ++j) {
    const int32_t first = chunk_first_seg[j];
    const int32_t last = (j + 1 < n_chunks ? chunk_first_seg[j + 1] : n_segments) - 1;
    const double d = (double)seg_end[last] - (double)seg_start[first];
    if (!(d >= 0.0)) return MURMUR_ERR_INVALID_ARG;
    const double s_tok = ceil(tokens_per_s * d);
    const double t_tok = d >= d_nominal ? (double)max_new_nominal : floor((double)max_new_nominal * d / d_nominal);
    const double total = (double)n_prefix + s_tok + (double)n_mid + (t_tok < 1.0 ? 1.0 : t_tok);
    if (!(total < 2147483647.0 - (double)page_size)) return MURMUR_ERR_INVALID_ARG;
    murmur_batch_entry_t e;
    e.chunk = j;
    e.batch = j / batch_size;
    e.slot = j % batch_size;
    e.n_speech = (int32_t)s_tok;
    e.max_new = t_tok < 1.0 ? 1 : (int32_t)t_tok;
    e.max_blocks = (int32_t)(((int64_t)n_prefix + e.n_speech + n_mid + e.max_new + page_size - 1) / page_size);
    entries[j] = e;
  }
  *n_batches_out = (n_chunks + batch_size - 1) / batch_size;
  return MURMUR_OK;
}
