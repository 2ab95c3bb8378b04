// murmur_kv_evict: apply the sliding-window policy at each sequence's current t.
//
// Alg. 1 line 3 / Alg. 2 line 6 "Evict {k_i, v_i | i not in K} from C",
// once per decode step.  With the position-paged layout (C2)
// nothing moves: a block whose every position is dead is pushed on the free stack
// (sequences in call order, blocks ascending - DESIGN.md C3), then the compacted live-page
// list, the run descriptors (maximal intervals of the retained set) and the attention tile
// list are rebuilt.  One CTA, one warp per sequence; the only cross-sequence dependency is
// the exclusive prefix sum of freed-block counts that fixes the push order.
#include "device_state.cuh"

namespace murmur {
namespace {

constexpr int kEvictThreads = 1024;
constexpr int kEvictWarps = kEvictThreads / 32;

__global__ void __launch_bounds__(kEvictThreads) evict_kernel(CacheView c, SeqList list) {
  __shared__ int s_ndead[kMaxSeqsPerLaunch];
  __shared__ int s_off[kMaxSeqsPerLaunch + 1];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const unsigned lt_mask = (1u << lane) - 1;
  const int n = list.n;
  const int free_top0 = c.ctrl[kCtrlFreeTop];
  const int p = c.p, plog = c.p_log2;

  // Phase 1: how many allocated blocks of each sequence are dead now.
  for (int i = warp; i < n; i += kEvictWarps) {
    const int id = list.ids[i];
    const SeqParams sp = load_params(c.seqs[id]);
    const int32_t* tab = c.block_table + (size_t)id * c.max_blocks;
    Interval dv[2];
    const int nd = c.seqs[id].active ? dead_intervals(sp, dv) : 0;
    int cnt = 0;
    for (int k = 0; k < nd; ++k) {
      int32_t lo, hi;
      blocks_inside(dv[k], p, &lo, &hi);
      for (int b = lo + lane; b < hi; b += 32) cnt += (tab[b] >= 0);
    }
    for (int o = 16; o > 0; o >>= 1) cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
    if (lane == 0) s_ndead[i] = cnt;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    int acc = 0;
    for (int i = 0; i < n; ++i) {
      s_off[i] = acc;
      acc += s_ndead[i];
    }
    s_off[n] = acc;
  }
  __syncthreads();

  // Phase 2: per sequence - push dead blocks, compact the table, rebuild runs and tiles.
  for (int i = warp; i < n; i += kEvictWarps) {
    const int id = list.ids[i];
    SeqDev& sd = c.seqs[id];
    if (!sd.active) continue;
    const SeqParams sp = load_params(sd);
    int32_t* tab = c.block_table + (size_t)id * c.max_blocks;
    int32_t* lpages = c.live_pages + (size_t)id * c.max_blocks;
    int32_t* lblocks = c.live_blocks + (size_t)id * c.max_blocks;

    Interval dv[2];
    const int nd = dead_intervals(sp, dv);
    int run = 0;
    const int base = free_top0 + s_off[i];
    for (int k = 0; k < nd; ++k) {
      int32_t lo, hi;
      blocks_inside(dv[k], p, &lo, &hi);
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
    __syncwarp();

    // compacted live-page list (stream compaction of the block table, ascending)
    const int nblk = (sp.len + p - 1) >> plog;
    int nl = 0;
    for (int b0 = 0; b0 < nblk; b0 += 32) {
      const int b = b0 + lane;
      const int pg = (b < nblk) ? tab[b] : -1;
      const unsigned m = __ballot_sync(0xffffffffu, pg >= 0);
      if (pg >= 0) {
        const int k = nl + __popc(m & lt_mask);
        lpages[k] = pg;
        lblocks[k] = b;
      }
      nl += __popc(m);
    }
    __syncwarp();

    // run descriptors: maximal intervals of A(t) + rank of their first block in the live list
    Interval rr[kMaxRuns];
    const int nr = retained_runs(sp, rr);
    if (lane < nr) {
      const int blk = rr[lane].a >> plog;
      int lo = 0, hi = nl - 1;  // binary search: lblocks ascending, blk is present
      while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if (lblocks[mid] < blk) lo = mid + 1; else hi = mid;
      }
      if (nl == 0 || lblocks[lo] != blk) atomicCAS(&c.ctrl[kCtrlError], 0, 2);
      sd.runs[lane][0] = rr[lane].a;
      sd.runs[lane][1] = rr[lane].b - rr[lane].a;
      sd.runs[lane][2] = lo;
    }
    __syncwarp();
    int n_ret = 0;
    for (int r = 0; r < nr; ++r) n_ret += rr[r].b - rr[r].a;

    // attention tiles: <= 64 consecutive rows of one run, made of 64/p consecutive live pages
    int n_tiles = 0;
    if (p >= 16 && p <= kTileRows) {
      const int ppt = kTileRows >> plog;  // pages per tile
      int toff[kMaxRuns + 1];
      toff[0] = 0;
      for (int r = 0; r < nr; ++r) {
        const int fb = rr[r].a >> plog, lb = (rr[r].b - 1) >> plog;
        toff[r + 1] = toff[r] + ((lb - fb + 1) + ppt - 1) / ppt;
      }
      n_tiles = toff[nr];
      TileDesc* tiles = c.tiles + (size_t)id * c.max_blocks;
      for (int tix = lane; tix < n_tiles; tix += 32) {
        int r = 0;
        while (tix >= toff[r + 1]) ++r;
        const int j = tix - toff[r];
        const int fb = rr[r].a >> plog, lb = (rr[r].b - 1) >> plog;
        const int b0 = fb + j * ppt;
        const int np = min(ppt, lb - b0 + 1);
        TileDesc td;
        td.n_pages = np;
        td.row_begin = (j == 0) ? (rr[r].a & (p - 1)) : 0;
        td.row_end = (b0 + np - 1 == lb) ? (np - 1) * p + ((rr[r].b - 1) & (p - 1)) + 1 : np * p;
        td.first_pos = (j == 0) ? rr[r].a : b0 * p;
        const int k0 = sd.runs[r][2] + j * ppt;
        for (int q = 0; q < 4; ++q) td.page[q] = (q < np) ? lpages[k0 + q] : -1;
        tiles[tix] = td;
      }
    }
    __syncwarp();
    if (lane == 0) {
      sd.n_live = nl;
      sd.n_runs = nr;
      sd.n_tiles = n_tiles;
      sd.n_retained = n_ret;
    }
  }
  if (threadIdx.x == 0) c.ctrl[kCtrlFreeTop] = free_top0 + s_off[n];
}

}  // namespace

cudaError_t launch_evict(const CacheView& c, const SeqList& list, cudaStream_t st, LaunchInfo* info) {
  evict_kernel<<<1, kEvictThreads, 0, st>>>(c, list);
  info->launches += 1;
  return cudaGetLastError();
}

}  // namespace murmur
