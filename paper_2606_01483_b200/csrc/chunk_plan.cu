// murmur_chunk_plan: greedy merge of VAD speech segments into chunks of at most max_len seconds.
//
// "Segments are greedily merged to construct chunks {C_1..C_m} where each chunk
// satisfies |C_i| <= c = 300 s"; the chunks are then submitted as one batch (the sequences of a
// murmur_decode_step call).  Host logic only - it runs once per recording, before any GPU work.
// Readings (G23): |C| is the span from the start of the chunk's first segment to the end
// of its last one (silences inside count: that audio is fed to the model); a single segment longer
// than max_len cannot be merged with anything and forms a chunk of its own.
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
