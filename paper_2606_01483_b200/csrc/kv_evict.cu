// murmur_kv_evict: apply the sliding-window policy at each sequence's current t.
//
// Alg. 1 line 3 / Alg. 2 line 6 "Evict {k_i, v_i | i not in K} from C",
// once per decode step.  With the position-paged layout (C2)
// nothing moves: a block whose every position is dead is pushed on the free stack
// (sequences in call order, blocks ascending - DESIGN.md C3), then the compacted live-page
// list, the run descriptors (maximal intervals of the retained set) and the attention tile
// list are rebuilt.  One CTA; the work is split into independent warp tasks (evict_body.cuh);
// the only cross-sequence dependency is the exclusive prefix sum of freed-block counts that
// fixes the push order.
#include "evict_body.cuh"

namespace murmur {
namespace {

constexpr int kEvictThreads = 1024;

__global__ void __launch_bounds__(kEvictThreads)
evict_kernel(const __grid_constant__ CacheView c, const __grid_constant__ SeqList list) {
  __shared__ int s_ndead[kMaxSeqsPerLaunch];
  __shared__ int s_off[kMaxSeqsPerLaunch + 1];
  __shared__ SeqParams s_sp[kMaxSeqsPerLaunch];
  pdl_launch_dependents();
  pdl_wait();
  const int free_top0 = c.ctrl[kCtrlFreeTop];
  for (int i = threadIdx.x; i < list.n; i += kEvictThreads) {
    const SeqDev& sd = c.seqs[list.ids[i]];
    s_sp[i] = load_params(sd);
    if (!sd.active) atomicCAS(&c.ctrl[kCtrlError], 0, 2);
  }
  __syncthreads();
  evict_body(c, list.ids, list.n, s_sp, free_top0, s_ndead, s_off);
}

}  // namespace

cudaError_t launch_evict(const CacheView& c, const SeqList& list, bool pdl, cudaStream_t st, LaunchInfo* info) {
  PdlLaunch l(dim3(1), dim3(kEvictThreads), 0, st, pdl);
  info->launches += 1;
  return cudaLaunchKernelEx(&l.cfg, evict_kernel, c, list);
}

}  // namespace murmur
