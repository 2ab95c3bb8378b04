// Body of murmur_kv_evict, shared by the stand-alone evict kernel (kv_evict.cu) and by the fused
// append+evict step prologue (kv_append.cu, last CTA).
//
// Alg. 1 line 3 / Alg. 2 line 6 "Evict {k_i, v_i | i not in K} from C",
// once per decode step.  With the position-paged layout (C2)
// nothing moves: a block whose every position is dead is pushed on the free stack
// (sequences in call order, blocks ascending - DESIGN.md C3), then the compacted live-page
// list, the run descriptors (maximal intervals of the retained set) and the attention tile
// list are rebuilt.
//
// Latency structure.  The dead positions form <= 2 intervals, hence the dead blocks <= 2 ascending
// block ranges [dlo_k, dhi_k), and every other block below nblk is live.  Ranks in the compacted
// list are therefore pure arithmetic and the three products of an evict - (0) the pages to free,
// (1) the compacted page list, (2) runs + tiles - do not depend on one another.  They are
// computed by independent warp tasks, each of which makes ONE round of block-table loads; only
// the push order (exclusive prefix sum of freed-block counts over the sequences) needs a
// CTA-wide synchronisation.  In the fused step prologue products 1 and 2 are spread over all the
// CTAs of the append kernel and only product 0 is left to its last CTA.  The table is still
// cross-checked: a live block without a page raises the device error word.
#pragma once
#include "device_state.cuh"

namespace murmur {

struct DeadRanges {
  int32_t lo0, hi0, lo1, hi1;  // [lo0, hi0) below [lo1, hi1); empty ranges have lo == hi
};

__device__ __forceinline__ DeadRanges dead_block_ranges(const SeqParams& sp, int plog) {
  Interval dv[2];
  const int n = dead_intervals(sp, dv);
  DeadRanges r;
  r.lo0 = r.hi0 = r.lo1 = r.hi1 = 0;
  if (n > 0) blocks_inside_log2(dv[0], plog, &r.lo0, &r.hi0);
  if (n > 1) blocks_inside_log2(dv[1], plog, &r.lo1, &r.hi1);
  return r;
}

// k-th live block (k-th block outside the dead ranges) and its inverse for a live block.
__device__ __forceinline__ int live_unrank(const DeadRanges& dr, int k) {
  int b = k;
  if (dr.hi0 > dr.lo0 && b >= dr.lo0) b += dr.hi0 - dr.lo0;
  if (dr.hi1 > dr.lo1 && b >= dr.lo1) b += dr.hi1 - dr.lo1;
  return b;
}
__device__ __forceinline__ int live_rank(const DeadRanges& dr, int blk) {
  return blk - max(0, min(dr.hi0, blk) - dr.lo0) - max(0, min(dr.hi1, blk) - dr.lo1);
}
__device__ __forceinline__ bool is_dead_block(const DeadRanges& dr, int blk) {
  return (blk >= dr.lo0 && blk < dr.hi0) || (blk >= dr.lo1 && blk < dr.hi1);
}

// Runs6 (device_state.cuh) of a sequence: same set as retained_runs() of policy_math.cuh.
__device__ __forceinline__ Runs6 retained_runs6(const SeqParams& s) {
  const int32_t t = seq_t(s);
  const int32_t l = mm_min(window_start(s, t), s.S);
  const int32_t B = s.P + s.S + s.M;
  const int32_t ra[6] = {0, s.P, s.P + l, s.P + s.S, B, B + mm_max(0, t - mm_min(s.w_o, t))};
  const int32_t rb[6] = {s.P, s.P + mm_min(s.k_s, s.S), s.P + window_end(s, l), B, B + mm_min(s.k_o, t), B + t};
  Runs6 r;
  r.mask = 0u;       // heads of merged groups
  unsigned member = 0u;  // non-empty slots absorbed by the group below them
  bool have = false;
  int32_t gb = 0;
#pragma unroll
  for (int i = 0; i < 6; ++i) {  // forward: same merge rule as retained_runs (touching or overlapping)
    r.a[i] = ra[i];
    r.b[i] = mm_min(rb[i], s.len);
    if (r.b[i] > r.a[i]) {
      if (have && r.a[i] <= gb) {
        member |= 1u << i;
        gb = mm_max(gb, r.b[i]);
      } else {
        r.mask |= 1u << i;
        gb = r.b[i];
        have = true;
      }
    }
  }
  int32_t carry = 0;  // positions are >= 0
#pragma unroll
  for (int i = 5; i >= 0; --i) {  // backward: a group's end is the max over its members
    if (member >> i & 1u) carry = mm_max(carry, r.b[i]);
    if (r.mask >> i & 1u) {
      r.b[i] = mm_max(r.b[i], carry);
      carry = 0;
    }
  }
  return r;
}

__device__ __forceinline__ TileGen make_tilegen(const SeqParams& sp, int p, int plog) {
  TileGen g;
  g.rr = retained_runs6(sp);
  const int ppt = kTileRows >> plog;  // pages per tile (tiles only exist for 16 <= p <= 64)
  g.n_tiles = 0;
  g.n_ret = 0;
#pragma unroll
  for (int i = 0; i < 6; ++i) {
    g.toff[i] = g.n_tiles;
    if (g.rr.mask >> i & 1u) {
      g.n_ret += g.rr.b[i] - g.rr.a[i];
      const int fb = g.rr.a[i] >> plog, lb = (g.rr.b[i] - 1) >> plog;
      g.n_tiles += ((lb - fb + 1) + ppt - 1) / ppt;
    }
  }
  if (p < 16 || p > kTileRows) g.n_tiles = 0;
  return g;
}

// Descriptor of tile tix (0 <= tix < n_tiles); page_of(b) maps a logical block to its page.
template <class Lookup>
__device__ __forceinline__ TileDesc tile_at(const TileGen& g, int tix, int p, int plog, const Lookup& page_of) {
  int32_t a = 0, b = 0, t0 = 0;
#pragma unroll
  for (int i = 0; i < 6; ++i)
    if ((g.rr.mask >> i & 1u) && tix >= g.toff[i]) { a = g.rr.a[i]; b = g.rr.b[i]; t0 = g.toff[i]; }
  const int ppt = kTileRows >> plog;
  const int j = tix - t0;
  const int fb = a >> plog, lb = (b - 1) >> plog;
  const int b0 = fb + j * ppt;
  const int np = min(ppt, lb - b0 + 1);
  TileDesc td;
  td.n_pages = np;
  td.row_begin = (j == 0) ? (a & (p - 1)) : 0;
  td.row_end = (b0 + np - 1 == lb) ? (np - 1) * p + ((b - 1) & (p - 1)) + 1 : np * p;
  td.first_pos = (j == 0) ? a : b0 * p;
#pragma unroll
  for (int q = 0; q < 4; ++q) td.page[q] = (q < np) ? page_of(b0 + q) : -1;
  return td;
}

// Page of logical block b of a sequence, as the eviction sees it.  The stand-alone kernel reads
// the block table; the fused step prologue, which runs these tasks BEFORE the append's integer
// state is committed, substitutes the pages the append is about to map (kv_append.cu).
struct TableLookup {
  const int32_t* tab;
  __device__ __forceinline__ int operator()(int b) const { return tab[b]; }
};

// One warp: product 1 (compacted live-page list) or product 2 (runs + tiles) of one sequence.
template <class Lookup>
__device__ __forceinline__ void evict_task(const CacheView& c, int id, const SeqParams& sp, int role, const Lookup& page_of) {
  const int lane = threadIdx.x & 31;
  const int p = c.p, plog = c.p_log2;
  const DeadRanges dr = dead_block_ranges(sp, plog);
  bool bad = false;
  if (role == 1) {
    // ---- compacted live-page list: entry k is the k-th block outside the dead ranges ----
    int32_t* lpages = c.live_pages + (size_t)id * c.max_blocks;
    int32_t* lblocks = c.live_blocks + (size_t)id * c.max_blocks;
    const int nblk = (sp.len + p - 1) >> plog;
    const int nl = nblk - (dr.hi0 - dr.lo0) - (dr.hi1 - dr.lo1);
    for (int k = lane; k < nl; k += 32) {
      const int b = live_unrank(dr, k);
      const int pg = page_of(b);
      bad |= (pg < 0);
      lpages[k] = pg;
      lblocks[k] = b;
    }
    if (lane == 0) c.seqs[id].n_live = nl;
  } else {
    // ---- run descriptors: maximal intervals of A(t) + rank of their first block in the live list ----
    SeqDev& sd = c.seqs[id];
    const TileGen g = make_tilegen(sp, p, plog);
    const Runs6& rr = g.rr;
    const int nr = __popc(rr.mask);
    const int n_tiles = g.n_tiles, n_ret = g.n_ret;
    if (lane < nr) {  // lane r writes run r = the r-th set slot
      const int slot = __fns(rr.mask, 0, lane + 1);
      int32_t a = 0, b = 0;
#pragma unroll
      for (int i = 0; i < 6; ++i)
        if (i == slot) { a = rr.a[i]; b = rr.b[i]; }
      const int blk = a >> plog;
      bad |= is_dead_block(dr, blk);
      sd.runs[lane][0] = a;
      sd.runs[lane][1] = b - a;
      sd.runs[lane][2] = live_rank(dr, blk);
    }
    // ---- attention tile list (read by tools; the attention kernel regenerates tiles itself) ----
    TileDesc* tiles = c.tiles + (size_t)id * c.max_blocks;
    for (int tix = lane; tix < n_tiles; tix += 32) {
      const TileDesc td = tile_at(g, tix, p, plog, page_of);
#pragma unroll
      for (int q = 0; q < 4; ++q) bad |= (q < td.n_pages) && (td.page[q] < 0);
      tiles[tix] = td;
    }
    if (lane == 0) {
      sd.n_runs = nr;
      sd.n_tiles = n_tiles;
      sd.n_retained = n_ret;
      // tile tables for the attention kernels: this length (unless already there - it may be in
      // use by concurrent readers, which never read an invalid slot) and the next decode step's
      SeqParams sp1 = sp;
      sp1.len += 1;
      sd.tg_len[sp1.len & 1] = -1;  // invalidate, then the table, then the length that validates it
      __threadfence();
      sd.tg[sp1.len & 1] = make_tilegen(sp1, p, plog);
      __threadfence();
      sd.tg_len[sp1.len & 1] = sp1.len;
      if (sd.tg_len[sp.len & 1] != sp.len) {
        sd.tg[sp.len & 1] = g;
        __threadfence();  // the table before the length that validates it
        sd.tg_len[sp.len & 1] = sp.len;
      }
    }
  }
  if (bad) atomicCAS(&c.ctrl[kCtrlError], 0, 2);
}

// Warp tasks: s_ndead[i] = mapped blocks inside the dead ranges of sequence i at length
// sp_sh[i].len (+ extra_len[i] if given).  With old_nblk (the fused append+evict prologue, which
// counts BEFORE the append's commit) the blocks [old_nblk[i], blocks at that length) count as mapped:
// the commit maps them before evict_free pushes (a block can be mapped and dead in the same step
// only when p == 1 and w_out == 0).
__device__ __forceinline__ void evict_count(const CacheView& c, const int32_t* ids, int n, const SeqParams* sp_sh,
                                            const int32_t* extra_len, int* s_ndead, const int* old_nblk = nullptr) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, n_warps = blockDim.x >> 5;
  for (int i = warp; i < n; i += n_warps) {
    SeqParams sp = sp_sh[i];
    if (extra_len != nullptr) sp.len += extra_len[i];
    const DeadRanges dr = dead_block_ranges(sp, c.p_log2);
    const int32_t* tab = c.block_table + (size_t)ids[i] * c.max_blocks;
    const int tab_end = old_nblk != nullptr ? old_nblk[i] : 0x7fffffff;  // blocks from here on: mapped by the pending commit
    int cnt = 0;
    for (int b = dr.lo0 + lane; b < dr.hi0; b += 32) cnt += (b >= tab_end) || (tab[b] >= 0);
    for (int b = dr.lo1 + lane; b < dr.hi1; b += 32) cnt += (b >= tab_end) || (tab[b] >= 0);
    for (int o = 16; o > 0; o >>= 1) cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
    if (lane == 0) s_ndead[i] = cnt;
  }
}

// CTA-wide: product 0.  Counts each sequence's newly dead (still mapped) blocks (unless the caller
// already has: `counted`), fixes the push order with an exclusive prefix sum in call order, pushes
// the pages (blocks ascending) and unmaps them.  sp_sh: SeqParams[n] in shared memory with the
// lengths as of this evict; s_ndead int[kMaxSeqsPerLaunch], s_off int[kMaxSeqsPerLaunch + 1] shared
// scratch; free_top0 = height of the free stack before this evict.  Must be called by every
// thread of the CTA.
__device__ __forceinline__ void evict_free(const CacheView& c, const int32_t* ids, int n, const SeqParams* sp_sh,
                                           int free_top0, int* s_ndead, int* s_off, bool counted = false) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, n_warps = blockDim.x >> 5;
  const unsigned lt_mask = (1u << lane) - 1;
  const int plog = c.p_log2;
  if (!counted) evict_count(c, ids, n, sp_sh, nullptr, s_ndead);
  __syncthreads();
  if (threadIdx.x == 0) {  // push order: sequences in call order
    int acc = 0;
    for (int i = 0; i < n; ++i) {
      s_off[i] = acc;
      acc += s_ndead[i];
    }
    s_off[n] = acc;
    c.ctrl[kCtrlFreeTop] = free_top0 + acc;
  }
  __syncthreads();
  for (int i = warp; i < n; i += n_warps) {
    if (s_ndead[i] == 0) continue;
    const DeadRanges dr = dead_block_ranges(sp_sh[i], plog);
    int32_t* tab = c.block_table + (size_t)ids[i] * c.max_blocks;
    int run = 0;
    const int base = free_top0 + s_off[i];
#pragma unroll
    for (int k = 0; k < 2; ++k) {
      const int lo = k ? dr.lo1 : dr.lo0, hi = k ? dr.hi1 : dr.hi0;
      for (int b0 = lo; b0 < hi; b0 += 32) {
        const int b = b0 + lane;
        const int pg = (b < hi) ? tab[b] : -1;
        const unsigned m = __ballot_sync(0xffffffffu, pg >= 0);
        if (pg >= 0) {
          c.free_stack[base + run + __popc(m & lt_mask)] = pg;
          tab[b] = -1;
        }
        run += __popc(m);
      }
    }
  }
}

// Product 0 by ONE warp (the keeper warp of the single-kernel decode step): sequences in call
// order, so the push offset is a running sum and no CTA-wide synchronisation is needed.
// len_sh[i] = the sequence's length as of this evict (regions and policy are read from SeqDev: they never change).
__device__ __forceinline__ void evict_free_warp(const CacheView& c, const int32_t* ids, int n, const int* len_sh,
                                                int free_top0) {
  const int lane = threadIdx.x & 31;
  const unsigned lt_mask = (1u << lane) - 1;
  int top = free_top0;
  for (int i = 0; i < n; ++i) {
    SeqParams sp = load_params(c.seqs[ids[i]]);
    sp.len = len_sh[i];
    const DeadRanges dr = dead_block_ranges(sp, c.p_log2);
    int32_t* tab = c.block_table + (size_t)ids[i] * c.max_blocks;
#pragma unroll
    for (int k = 0; k < 2; ++k) {
      const int lo = k ? dr.lo1 : dr.lo0, hi = k ? dr.hi1 : dr.hi0;
      for (int b0 = lo; b0 < hi; b0 += 32) {
        const int b = b0 + lane;
        const int pg = (b < hi) ? tab[b] : -1;
        const unsigned m = __ballot_sync(0xffffffffu, pg >= 0);
        if (pg >= 0) {
          c.free_stack[top + __popc(m & lt_mask)] = pg;
          tab[b] = -1;
        }
        top += __popc(m);
      }
    }
  }
  if (lane == 0) c.ctrl[kCtrlFreeTop] = top;
}

// Product 0 of a decode step, the short way.  When everything that was dead at length - 1 has been freed (the
// caller knows: an evict or a step ran there), the pages to free at `len` are the blocks inside the dead ranges
// at len that were outside the dead ranges at len - 1 - the windows move a few positions per step, so that is
// 0..2 blocks per sequence.  One THREAD looks up one sequence (kFreeCand block-table loads, all independent), so a
// warp has the candidates of 64 sequences after one round trip, where evict_free_warp makes two per sequence.
constexpr int kFreeCand = 4;
struct FreeCand {
  int32_t b[kFreeCand], pg[kFreeCand];  // newly dead blocks (ascending) and their pages (-1: not mapped)
  int32_t n;                            // pages to push
};

// Returns false when the short way does not apply to sequence i (table not ready, or more than kFreeCand newly dead
// blocks): the caller then runs evict_free_warp for the whole call.  i >= n gives an empty candidate list.
// old_nblk / newpage: the block this step's commit maps (it may be written to the table concurrently).
__device__ __forceinline__ bool free_candidates(const CacheView& c, const int32_t* ids, int n, int i, const int* len_sh,
                                                const uint8_t* flags, const int* old_nblk, const int* newpage,
                                                FreeCand& fc) {
#pragma unroll
  for (int k = 0; k < kFreeCand; ++k) fc.b[k] = fc.pg[k] = -1;
  fc.n = 0;
  if (i >= n) return true;
  if (!(flags[i] & 2)) return false;
  SeqParams sp = load_params(c.seqs[ids[i]]);
  sp.len = len_sh[i];
  const DeadRanges dn = dead_block_ranges(sp, c.p_log2);
  sp.len -= 1;
  const DeadRanges dold = dead_block_ranges(sp, c.p_log2);
  int cnt = 0;
  bool ok = true;
#pragma unroll
  for (int r = 0; r < 2; ++r) {
    const int hi = r ? dn.hi1 : dn.hi0;
    int b = r ? dn.lo1 : dn.lo0;
    while (b < hi) {
      if (b >= dold.lo0 && b < dold.hi0) { b = dold.hi0; continue; }
      if (b >= dold.lo1 && b < dold.hi1) { b = dold.hi1; continue; }
      if (cnt == kFreeCand) { ok = false; break; }
#pragma unroll
      for (int k = 0; k < kFreeCand; ++k)
        if (k == cnt) fc.b[k] = b;
      ++cnt;
      ++b;
    }
  }
  if (!ok) return false;
  const int32_t* tab = c.block_table + (size_t)ids[i] * c.max_blocks;
#pragma unroll
  for (int k = 0; k < kFreeCand; ++k) {
    const int b = fc.b[k];
    if (b >= 0) fc.pg[k] = b < old_nblk[i] ? tab[b] : (b == old_nblk[i] ? newpage[i] : -1);
  }
#pragma unroll
  for (int k = 0; k < kFreeCand; ++k) fc.n += fc.pg[k] >= 0;
  return true;
}

// Pushes the candidates of sequence i at free_stack[at ...] and unmaps them (i may be past the list: fc.n == 0).
__device__ __forceinline__ void free_push(const CacheView& c, const int32_t* ids, int i, const FreeCand& fc, int at) {
  if (fc.n == 0) return;
  int32_t* tab = c.block_table + (size_t)ids[i] * c.max_blocks;
#pragma unroll
  for (int k = 0; k < kFreeCand; ++k) {
    if (fc.pg[k] >= 0) {
      c.free_stack[at++] = fc.pg[k];
      tab[fc.b[k]] = -1;
    }
  }
}

// The whole eviction in one CTA (stand-alone kernel).
__device__ __forceinline__ void evict_body(const CacheView& c, const int32_t* ids, int n, const SeqParams* sp_sh,
                                           int free_top0, int* s_ndead, int* s_off) {
  const int warp = threadIdx.x >> 5, n_warps = blockDim.x >> 5;
  if (threadIdx.x == 0) step_stamp(c, 3);
  for (int task = warp; task < 2 * n; task += n_warps) {
    const int role = 1 + task / n, i = task % n;
    const TableLookup lk{c.block_table + (size_t)ids[i] * c.max_blocks};
    evict_task(c, ids[i], sp_sh[i], role, lk);
  }
  evict_free(c, ids, n, sp_sh, free_top0, s_ndead, s_off);
  if (threadIdx.x == 0) step_stamp(c, 4);
}

}  // namespace murmur
