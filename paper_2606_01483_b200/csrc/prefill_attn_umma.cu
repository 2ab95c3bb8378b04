// murmur_prefill_attn on the 5th-generation tensor cores: tcgen05.mma with accumulators in tensor memory.
//
// PAPER.md:95 (chunks are submitted to the engine, which first runs prompt + speech tokens through the
// model) and PAPER.md:77 (prefill = what is left of model time after the 95.3 % of decoding).  Position
// x attends, by Eq. 1, to the cache positions y <= x.  This is the one dense
// contraction of the path, so it runs where dense contractions belong on sm_100a.
//
// Work item = a PAIR of row blocks of the same (layer, KV head); a row block is 128 consecutive query
// positions of one query head.  Row blocks are enumerated with the head of the GQA group fastest, so the two
// blocks of a pair nearly always cover the SAME query positions for two heads that share K/V: every 128-key
// K/V tile is staged once and used by both (M = 256 rows per staged tile).
//
// PERSISTENT CTAs, one per SM: items are ordered layer by layer (K/V of a layer or two stay in L2), heaviest pair
// first inside a layer, and dealt round-robin - CTA c takes items c, c + grid, c + 2 grid, ...  All barriers and the
// K/V ring run on across items: while the softmax warps finish an item (last tiles, O / l -> out), the producer
// already streams the next item's Q and K/V and the issuer its first score tiles.  (One CTA per item cost ~10 us of
// launch, set-up, pipeline fill and drain per item - as much as the item's tensor-core time.)
//
// Per CTA, 24 warps in six warpgroups (register budgets re-balanced with setmaxnreg):
//   warp 0      TMA producer: Q blocks (tensor map over q, 128-byte swizzle written by the copy engine) and
//               the K/V tiles, one box per (page, d-half) straight from the paged pools.  The pools' rows are
//               stored pre-swizzled (16-byte chunk c of slot s at c ^ (s & 7), device_state.cuh); a
//               [p slots][64 bf16] box of one d-half therefore lands as exactly the 128-byte-swizzled tile
//               image tcgen05.mma expects - the decode kernels' layout needs no re-tiling.
//   warp 1      MMA issuer: S_w = Q_w K^T (SS, both operands K-major) and O_w += P_w V (A = P from tensor memory,
//               B = V MN-major), completion signalled with tcgen05.commit.  Issue order per tile j:
//               S(1,j)  PV(0,j)  S(0,j+1)  PV(1,j) - the two row blocks run half a period apart, so one block's
//               softmax has the other's MMAs to hide under.  tcgen05.mma issue does not run ahead of the tensor
//               pipe: every instruction executed between two MMAs is tensor-pipe idle time (profiles/
//               r02_prefill_ncu.md, rate probes).  The whole warp walks the loop (all warp-uniform, so descriptors
//               and tensor-memory addresses are formed on the uniform datapath) and one elected lane issues.
//   warps 2-3   idle (they fill the issuer's warpgroup; setmaxnreg is per warpgroup)
//   warps 4-19  softmax: 16 warps serve BOTH row blocks, tile by tile in issue order.  Four warps per tensor-memory
//               lane quarter; warp `cq` of a quarter owns key columns [32 cq, 32 cq + 32) of every row of the quarter:
//               tcgen05.ld, causal mask on the diagonal, row maximum (exchanged through shared memory), exp2 (part
//               of it on the FMA pipes), P written back as bf16 over the first 16 of the thread's OWN 32 score
//               columns (tcgen05.st).  The reference maximum is raised only when it grows by more than 2^8 (O is
//               then rescaled in tensor memory): rare, and exact in the end - l and O share one reference.
//   warps 20-23 epilogue, one per lane quarter: O_w / l -> bf16 -> 4 KB staging slice -> TMA store, while the
//               softmax warps are already on the next item's first tiles.
// Tensor memory (512 columns): S_0, S_1 (128 fp32 columns each, P_w inside S_w), O_0, O_1.
#include <cuda_bf16.h>

#include <type_traits>

#include "device_state.cuh"
#include "ptx_utils.cuh"
#include "umma_utils.cuh"

namespace murmur {
namespace {

constexpr int kBM = 128;                      // query rows per row block (TMEM lanes)
constexpr int kBN = 128;                      // keys per K/V tile
constexpr int kHalfBytes = kBN * 128;         // one d-half of a 128-row tile: [128][64 bf16] = 16 KB
constexpr int kUStages = 2;
constexpr int kUThreads = 768;                // 6 warpgroups: {producer, issuer, 2 idle}, 4 x softmax, epilogue
constexpr int kSoftmaxWarps = 16;
constexpr uint32_t kTmemCols = 512;
constexpr float kRescaleLog2 = 8.f;           // raise the reference maximum only past 2^8
constexpr int kRegsSoftmax = 88, kRegsOther = 48, kRegsEpilogue = 72;  // 512 x 88 + 128 x 48 + 128 x 72 = 60416 <= 768 x 80 (what the launch allocates)

struct __align__(1024) USmem {
  uint8_t q[2][2][kHalfBytes];                // [row block][d-half]
  uint8_t k[kUStages][2][kHalfBytes];         // [stage][d-half]
  uint8_t v[kUStages][2][kHalfBytes];
  uint8_t ostage[4][32 * 128];                // per lane quarter: [32 rows][64 bf16] of one d-half on its way out (TMA store)
  float mxch[2][4][kBM];                      // row maxima of the four warps of a row, [exchange parity]
  float lfin[2][2][4][kBM], mfin[2][2][kBM];  // an item's row sums (four partials) and reference maxima on their way to the epilogue, [item parity][row block]
  unsigned long long q_full[2], q_empty[2], k_full[kUStages], v_full[kUStages], k_empty[kUStages], v_empty[kUStages];
  unsigned long long s_ready[2], p_ready[2], o_done[2], o_free[2], l_ready[2], l_free[2], v_clean[2], xch[4];
  uint32_t tmem_base;
};

struct UParams {
  uint16_t* out;   // [layers][n_tok][n_q][128]
  float* lse;      // [layers][n_tok][n_q] or null
  int seq, pos_begin, n_tok, layer_begin;
  float sm_scale;
};

// One work item, derived from its index by every role on its own (integer arithmetic only).
struct Item {
  int lc, kvh, act[2], hq[2], x0[2], xl[2], nkt[2], n_kt, x_last, first_bad;
  bool need_clean;
};
__device__ __forceinline__ Item make_item(int id, const CacheView& c, const UParams& prm, int len) {
  Item it;
  const int G = c.group;
  const int n_qb = (prm.n_tok + kBM - 1) / kBM;
  const int n_rb = n_qb * G;                  // row blocks of a (layer, KV head): e = b * G + g
  const int n_pairs = (n_rb + 1) >> 1;
  const int per_layer = n_pairs * c.n_kv;
  it.lc = id / per_layer;
  const int r = id - it.lc * per_layer;
  const int pair = n_pairs - 1 - r / c.n_kv;  // heaviest (latest queries) first
  it.kvh = r % c.n_kv;
  const int pos_end = prm.pos_begin + prm.n_tok;
#pragma unroll
  for (int w = 0; w < 2; ++w) {
    const int e = 2 * pair + w;
    it.act[w] = e < n_rb;
    const int b = it.act[w] ? e / G : 0;
    it.hq[w] = it.kvh * G + (it.act[w] ? e % G : 0);
    it.x0[w] = prm.pos_begin + b * kBM;
    it.xl[w] = min(pos_end, it.x0[w] + kBM) - 1;
    it.nkt[w] = it.act[w] ? (it.xl[w] >> 7) + 1 : 0;
  }
  it.n_kt = max(it.nkt[0], it.nkt[1]);
  it.x_last = max(it.xl[0], it.act[1] ? it.xl[1] : 0);
  // rows at or beyond the sequence length (inside the last mapped page) hold whatever the pool holds: their P is
  // 0, but 0 * NaN would poison O - the producer warp zeroes them in the item's last tile before PV may read it
  it.first_bad = len - (it.n_kt - 1) * kBN;
  it.need_clean = it.first_bad < kBN;
  return it;
}

// packed fp32 pairs (sm_100a): halve the FFMA / FADD issue slots of the softmax
__device__ __forceinline__ unsigned long long pack2f(float lo, float hi) {
  unsigned long long r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
  return r;
}
__device__ __forceinline__ void unpack2f(unsigned long long v, float& lo, float& hi) {
  asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ unsigned long long ffma2(unsigned long long a, unsigned long long b, unsigned long long c) {
  unsigned long long d;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
  return d;
}
__device__ __forceinline__ unsigned long long fadd2(unsigned long long a, unsigned long long b) {
  unsigned long long d;
  asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
  return d;
}

// exp2 of a packed pair on the FMA pipes (the SFUs do 16 exp2 per clock and SM: as many cycles per 128-key tile
// as its two MMA groups, so part of the exponentials is taken off them): x = n + f with n = round(x), f in
// [-1/2, 1/2]; 2^f by a cubic (minimax in relative error, 7.5e-5 - P is rounded to bf16, 2^-9, right after);
// 2^n by adding n to the exponent field.  x + 1.5 * 2^23 leaves round(x) in the low mantissa bits.
__device__ __forceinline__ unsigned long long ex2_fma2(unsigned long long x2) {
  float x0, x1;
  unpack2f(x2, x0, x1);
  const unsigned long long xc = pack2f(fmaxf(x0, -125.f), fmaxf(x1, -125.f));  // keeps 2^n normal (and -inf finite)
  const unsigned long long magic = pack2f(12582912.f, 12582912.f);
  const unsigned long long t = fadd2(xc, magic);
  const unsigned long long nf = fadd2(t, pack2f(-12582912.f, -12582912.f));
  const unsigned long long f = ffma2(nf, pack2f(-1.f, -1.f), xc);
  unsigned long long q = ffma2(f, pack2f(0.05517132207751274f, 0.05517132207751274f), pack2f(0.24261054396629333f, 0.24261054396629333f));
  q = ffma2(q, f, pack2f(0.6932609677314758f, 0.6932609677314758f));
  q = ffma2(q, f, pack2f(0.9999281167984009f, 0.9999281167984009f));
  float q0, q1, t0, t1;
  unpack2f(q, q0, q1);
  unpack2f(t, t0, t1);
  return pack2f(__uint_as_float(__float_as_uint(q0) + (__float_as_uint(t0) << 23)),
                __uint_as_float(__float_as_uint(q1) + (__float_as_uint(t1) << 23)));
}
#ifndef MURMUR_PF_EMU_OF_8
#define MURMUR_PF_EMU_OF_8 1
#endif
constexpr int kEmuOf8 = MURMUR_PF_EMU_OF_8;   // of every 8 pairs, this many take the FMA route

#ifdef MURMUR_PFTRACE
// Profiling builds only (-DMURMUR_PFTRACE): per-item clock stamps of CTA 0's issuer warp and softmax warp 4.
__device__ long long g_pftrace[2][8192];
#define PFT(role, idx) do { if (blockIdx.x == 0 && lane == 0 && (idx) < 8192) g_pftrace[role][idx] = clock64(); } while (0)
#define PFV(role, idx, v) do { if (blockIdx.x == 0 && lane == 0 && (idx) < 8192) g_pftrace[role][idx] = (v); } while (0)
__device__ long long g_pftile[3][1024];
constexpr int kTraceItem = 2;
#define PFD(cond, role, idx) do { if (blockIdx.x == 0 && lane == 0 && (cond) && (idx) < 1024) g_pftile[role][idx] = clock64(); } while (0)
#else
#define PFD(cond, role, idx) do { } while (0)
#define PFT(role, idx) do { } while (0)
#define PFV(role, idx, v) do { } while (0)
#endif

template <int N>
__device__ __forceinline__ void set_regs_inc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(N)); }
template <int N>
__device__ __forceinline__ void set_regs_dec() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(N)); }

__global__ void __launch_bounds__(kUThreads, 1)
prefill_umma_kernel(const __grid_constant__ CUtensorMap tm_q, const __grid_constant__ CUtensorMap tm_k,
                    const __grid_constant__ CUtensorMap tm_v, const __grid_constant__ CUtensorMap tm_o,
                    const __grid_constant__ CacheView c, const __grid_constant__ UParams prm, const int n_items) {
  extern __shared__ uint8_t smem_raw[];
  USmem& s = *reinterpret_cast<USmem*>(smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u));
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int p = c.p, plog = c.p_log2;
  const int len = c.seqs[prm.seq].len;
  const int first = (int)blockIdx.x, stride = (int)gridDim.x;

  // ---- set-up: barriers, tensor memory, finite K/V stages ------------------------------------------
  if (tid == 0) {
    for (int w = 0; w < 2; ++w) {
      mbar_init(&s.q_full[w], 1);
      mbar_init(&s.q_empty[w], 1);
    }
    for (int i = 0; i < kUStages; ++i) {
      mbar_init(&s.k_full[i], 1);
      mbar_init(&s.v_full[i], 1);
      mbar_init(&s.k_empty[i], 1);
      mbar_init(&s.v_empty[i], 1);
    }
    for (int w = 0; w < 2; ++w) {
      mbar_init(&s.s_ready[w], 1);
      mbar_init(&s.p_ready[w], kSoftmaxWarps);  // one arrival per softmax warp
      mbar_init(&s.o_done[w], 1);
      mbar_init(&s.o_free[w], 4);               // the four epilogue warps
      mbar_init(&s.l_ready[w], kSoftmaxWarps);
      mbar_init(&s.l_free[w], 4);               // the four epilogue warps
      mbar_init(&s.v_clean[w], 1);
    }
    for (int i = 0; i < 4; ++i) mbar_init(&s.xch[i], 4);  // the four warps of a lane quarter
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    tma_prefetch_desc(&tm_q);
    tma_prefetch_desc(&tm_k);
    tma_prefetch_desc(&tm_v);
    tma_prefetch_desc(&tm_o);
  }
  if (warp == 1) {
    tmem_alloc(&s.tmem_base, kTmemCols);
    tmem_relinquish();
  }
  // rows of a partial last tile that no copy writes must still be finite (P = 0 times NaN is NaN); later tiles
  // find older, finite, K/V rows there
  for (int i = tid; i < (int)(sizeof(s.v) / 16); i += kUThreads) reinterpret_cast<uint4*>(&s.v[0][0][0])[i] = make_uint4(0u, 0u, 0u, 0u);
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  // All 512 columns are ours, so the allocation starts at lane 0 / column 0; using the literal (checked here)
  // keeps the tcgen05 operands provably warp-uniform for the compiler.
  if (s.tmem_base != 0u) {
    if (tid == 0) atomicCAS(&c.ctrl[kCtrlError], 0, 4);
    __trap();
  }
  constexpr uint32_t tb = 0u;

  if (warp < 4) {
    set_regs_dec<kRegsOther>();
    if (warp == 0) {
      // ============================== TMA producer ==============================
      const int32_t* tab = c.block_table + (size_t)prm.seq * c.max_blocks;
      const int ppt = kBN >> plog;  // pages per tile
      int t = 0;                    // K/V tiles staged so far (ring position, across items)
      uint32_t n_it = 0, n_qw[2] = {0u, 0u};   // items; items with row block w active (parity of q_empty[w])
      uint32_t n_clean = 0;                    // tiles cleaned so far
      for (int id = first; id < n_items; id += stride, ++n_it) {
        const Item it = make_item(id, c, prm, len);
        const int layer = prm.layer_begin + it.lc;
        if (lane == 0) {
          auto stage_tile = [&](int j) {
            const int st = t % kUStages;
            const uint32_t ph = (uint32_t)(t / kUStages) & 1u;
            mbar_wait(&s.k_empty[st], ph ^ 1u);
            const int rows = min(kBN, it.x_last + 1 - j * kBN);   // keys beyond x_last are never needed
            const int pages = (rows + p - 1) >> plog;             // whole pages (all mapped: x_last < len)
            const uint32_t bytes = (uint32_t)pages * (uint32_t)p * kRowBytes;
            mbar_expect_tx(&s.k_full[st], bytes);
            for (int pg = 0; pg < pages; ++pg) {
              const int page = tab[j * ppt + pg];
              for (int h = 0; h < 2; ++h) tma_load_5d(&s.k[st][h][pg * p * 128], &tm_k, 64 * h, 0, it.kvh, page, layer, &s.k_full[st]);
            }
            mbar_wait(&s.v_empty[st], ph ^ 1u);
            mbar_expect_tx(&s.v_full[st], bytes);
            for (int pg = 0; pg < pages; ++pg) {
              const int page = tab[j * ppt + pg];
              for (int h = 0; h < 2; ++h) tma_load_5d(&s.v[st][h][pg * p * 128], &tm_v, 64 * h, 0, it.kvh, page, layer, &s.v_full[st]);
            }
            ++t;
          };
          // Q_w has its own hand-over: the previous item's last score tile of row block w frees it - for row block 0
          // that is two MMA groups before the item ends, so Q_0 and the first K/V tile (the ring slot frees at about
          // the same time) are there for the successor's first score tile to be issued under the tail
          auto load_q = [&](int w) {
            if (!it.act[w]) return;
            mbar_wait(&s.q_empty[w], (n_qw[w] & 1u) ^ 1u);
            ++n_qw[w];
            mbar_expect_tx(&s.q_full[w], (uint32_t)(2 * kHalfBytes));
            for (int h = 0; h < 2; ++h)
              tma_load_4d(&s.q[w][h][0], &tm_q, 64 * h, it.hq[w], it.x0[w] - prm.pos_begin, it.lc, &s.q_full[w]);
          };
          load_q(0);
          stage_tile(0);
          load_q(1);
          if (id + stride < n_items) {  // the NEXT item's Q on its way into L2 (it comes from HBM: q is read once)
            const Item nx = make_item(id + stride, c, prm, len);
#pragma unroll
            for (int w = 0; w < 2; ++w)
              if (nx.act[w])
                for (int h = 0; h < 2; ++h) tma_prefetch_4d(&tm_q, 64 * h, nx.hq[w], nx.x0[w] - prm.pos_begin, nx.lc);
          }
          for (int j = 1; j < it.n_kt; ++j) stage_tile(j);
        }
        t = __shfl_sync(0xffffffffu, t, 0);
        if (it.need_clean) {  // the whole warp: zero the V rows at / beyond the sequence length in the item's last tile
          const int tl = t - 1, st = tl % kUStages;
          mbar_wait(&s.v_full[st], (uint32_t)(tl / kUStages) & 1u);
          const int fb = max(it.first_bad, 0);
          for (int i = lane; i < (kBN - fb) * 16; i += 32) {
            const int r = fb + (i >> 4), ch = i & 15;
            *reinterpret_cast<uint4*>(&s.v[st][ch >> 3][r * 128 + (ch & 7) * 16]) = make_uint4(0u, 0u, 0u, 0u);
          }
          asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
          __syncwarp();
          // two barriers in turn: the producer is at most two tiles - two cleaned tiles - ahead of the issuer, so
          // neither barrier ever runs two phases ahead of its waiter (a parity wait could not tell)
          if (lane == 0) mbar_arrive(&s.v_clean[n_clean & 1u]);
          ++n_clean;
        }
      }
    } else if (warp == 1) {
      // ============================== MMA issuer ==============================
      const bool leader = elect_one();
      constexpr uint32_t idesc_s = umma_idesc_bf16(kBM, kBN, 0, 0);   // S = Q K^T: A, B K-major
      constexpr uint32_t idesc_o = umma_idesc_bf16(kBM, 128, 0, 1);   // O += P V: A from TMEM, B (V) MN-major, N = d = 128
      // One descriptor per operand array; tiles, d-halves and k-steps only add to the 14-bit start-address field
      // (16-byte units; everything lives below 256 KB, so no carry leaves the field).
      const uint64_t qd = smem_desc_kmajor(smem_u32(&s.q[0][0][0]));
      const uint64_t kd = smem_desc_kmajor(smem_u32(&s.k[0][0][0]));
      const uint64_t vd = smem_desc_mnmajor(smem_u32(&s.v[0][0][0]), kHalfBytes);
      constexpr uint32_t kHalfU = kHalfBytes >> 4, kTileU = 2 * kHalfU;
      int t0 = 0;                        // ring position of the current item's tile 0
      int k_seen = -1, v_seen = -1;      // ring positions whose full barrier this warp has already observed
      uint32_t n_pv[2] = {0u, 0u};       // PV groups issued per row block (parity of p_ready)
      uint32_t n_it = 0, n_itw[2] = {0u, 0u}, n_clean = 0;
      uint32_t n_qw[2] = {0u, 0u};       // items with row block w active whose Q this warp has taken (parity of q_full[w])
      bool s00_early = false;            // this item's S(0,0) was already issued under the previous item's tail
      for (int id = first; id < n_items; id += stride, ++n_it) {
        const Item it = make_item(id, c, prm, len);
        auto need_k = [&](int j) {
          const int t = t0 + j;
          if (k_seen < t) {
            mbar_wait(&s.k_full[t % kUStages], (uint32_t)(t / kUStages) & 1u);
            k_seen = t;
          }
        };
        auto need_v = [&](int j) {
          const int t = t0 + j;
          if (v_seen < t) {
            mbar_wait(&s.v_full[t % kUStages], (uint32_t)(t / kUStages) & 1u);
            if (it.need_clean && j == it.n_kt - 1) mbar_wait(&s.v_clean[n_clean & 1u], (n_clean >> 1) & 1u), ++n_clean;
            v_seen = t;
          }
        };
        auto issue_s = [&](auto wc, int j) {  // S_w = Q_w K_j^T
          constexpr int w = decltype(wc)::value;
          need_k(j);
          tc_fence_after();
          const uint64_t qa = qd + (uint32_t)w * kTileU, ka = kd + (uint32_t)((t0 + j) % kUStages) * kTileU;
          PFD(n_it == kTraceItem, 0, 16 * j + (w ? 0 : 6));
          if (leader) {
#pragma unroll
            for (int kk = 0; kk < 8; ++kk)  // +32 bytes per k-step inside a d-half, +16 KB for the second d-half
              umma_ss(tb + 128u * w, qa + (kk >> 2) * kHalfU + 2u * (kk & 3), ka + (kk >> 2) * kHalfU + 2u * (kk & 3), idesc_s, kk ? 1u : 0u);
            umma_commit(&s.s_ready[w]);
          }
          __syncwarp();
          PFD(n_it == kTraceItem, 0, 16 * j + (w ? 0 : 6) + 1);
        };
        auto issue_pv = [&](auto wc, int j) {  // O_w += P_w V_j
          constexpr int w = decltype(wc)::value;
          need_v(j);
          const uint64_t va = vd + (uint32_t)((t0 + j) % kUStages) * kTileU;
          if (j == 0) {  // the first PV of the item overwrites O_w: the previous item's epilogue must have read it
            mbar_wait(&s.o_free[w], (n_itw[w] & 1u) ^ 1u);
            ++n_itw[w];
          }
          PFD(n_it == kTraceItem, 0, 16 * j + (w ? 8 : 2));
          mbar_wait(&s.p_ready[w], n_pv[w] & 1u);
          ++n_pv[w];
          tc_fence_after();
          PFD(n_it == kTraceItem, 0, 16 * j + (w ? 8 : 2) + 1);
          if (leader) {
#pragma unroll
            for (int kk = 0; kk < 8; ++kk)  // 16 keys per instruction: P of keys 32 c .. 32 c + 31 at columns 32 c .. 32 c + 15; V rows 16 kk.. (+2048 bytes = +128)
              umma_ts(tb + 256u + 128u * w, tb + 128u * w + 32u * (kk >> 1) + 8u * (kk & 1), va + 128u * kk, idesc_o, (j | kk) ? 1u : 0u);
            umma_commit(&s.o_done[w]);
          }
          __syncwarp();
          PFD(n_it == kTraceItem, 0, 16 * j + 12 + w);
        };
        constexpr std::integral_constant<int, 0> W0{};
        constexpr std::integral_constant<int, 1> W1{};
        PFT(0, 8 * n_it + 0);
        PFV(0, 8 * n_it + 3, it.n_kt);
        // Issue order (the two row blocks half a period apart, so that one block's softmax always runs
        // under the other's MMAs):  S(0,0);  then per tile j:  S(1,j)  PV(0,j)  S(0,j+1)  PV(1,j).
        // P_w lives inside S_w: S(w,j+1) is issued after PV(w,j), and tcgen05.mma executes in issue order.
        // Row block 0 always exists (e = 2 pair < n_rb).
        if (!s00_early) {
          mbar_wait(&s.q_full[0], n_qw[0] & 1u);
          issue_s(W0, 0);
        }
        s00_early = false;
        ++n_qw[0];
        if (it.nkt[0] == 1) {
          if (leader) umma_commit(&s.q_empty[0]);  // that was row block 0's last score tile of the item: Q_0 may go
          __syncwarp();
        }
        PFT(0, 8 * n_it + 1);
        const bool has_next = id + stride < n_items;
        for (int j = 0; j < it.n_kt; ++j) {
          const int st = (t0 + j) % kUStages;
          if (j < it.nkt[1]) {
            if (j == 0) {
              mbar_wait(&s.q_full[1], n_qw[1] & 1u);
              ++n_qw[1];
            }
            issue_s(W1, j);
          }
          if (leader) {
            umma_commit(&s.k_empty[st]);  // K_j: both S(0,j) and S(1,j) are behind this point
            if (j == it.nkt[1] - 1) umma_commit(&s.q_empty[1]);
          }
          __syncwarp();
          if (j < it.nkt[0]) issue_pv(W0, j);
          if (j + 1 < it.nkt[0]) {
            issue_s(W0, j + 1);
            if (j + 1 == it.nkt[0] - 1) {
              if (leader) umma_commit(&s.q_empty[0]);
              __syncwarp();
            }
          } else if (j == it.n_kt - 1 && has_next) {
            // the slot of S(0, j+1) in the item's last round: the NEXT item's S(0,0) - its pipeline fills under this item's tail
            // (both waits end without this warp's help: the producer was handed Q_0 and the ring slot a round ago;
            // PV(1, j) behind them has the softmax of (1, j) to wait for anyway)
            mbar_wait(&s.q_full[0], n_qw[0] & 1u);
            issue_s(W0, it.n_kt);   // ring tile t0 + n_kt = the next item's tile 0
            s00_early = true;
          }
          if (j < it.nkt[1]) issue_pv(W1, j);
          if (leader) umma_commit(&s.v_empty[st]);
          __syncwarp();
        }
        t0 += it.n_kt;
        PFT(0, 8 * n_it + 2);
      }
    }
  } else if (warp < 4 + kSoftmaxWarps) {
    // ============================== softmax warps ==============================
    set_regs_inc<kRegsSoftmax>();
    const int sw = warp - 4;
    const int cq = sw >> 2;                // key-column quarter of this warp
    const int q4 = warp & 3;               // TMEM lane quarter this warp may access
    const int row = q4 * 32 + lane;
    const uint32_t lane_base = tb + ((uint32_t)(q4 * 32) << 16);
    const float c2 = prm.sm_scale * 1.4426950408889634f;
    const unsigned long long c2p = pack2f(c2, c2);
    uint32_t n_s[2] = {0u, 0u};            // score tiles consumed per row block (barrier parities)
    [[maybe_unused]] uint32_t n_done = 0;
    uint32_t n_x = 0;                      // maximum exchanges of this lane quarter so far (parity of xch)
    uint32_t n_fin[2] = {0u, 0u};          // items handed to the epilogue per row block (parity of lfin / mfin)
    for (int id = first; id < n_items; id += stride) {
      const Item it = make_item(id, c, prm, len);
      float m_[2] = {-INFINITY, -INFINITY};
      unsigned long long l_[2] = {pack2f(0.f, 0.f), pack2f(0.f, 0.f)};

      auto tile = [&](auto wc, int j) {
        constexpr int w = decltype(wc)::value;
        float& m = m_[w];
        unsigned long long& l2 = l_[w];
        const int x = it.x0[w] + row;                                      // this thread's query position
        const uint32_t s_addr = lane_base + 128u * w + 32u * cq;           // this thread's 32 score columns
        const uint32_t o_addr = lane_base + 256u + 128u * w + 32u * cq;    // this thread's quarter of the O row
        PFD(n_done == kTraceItem && warp == 4, 1 + w, 8 * j + 0);
        mbar_wait(&s.s_ready[w], n_s[w] & 1u);
        ++n_s[w];
        tc_fence_after();
        PFD(n_done == kTraceItem && warp == 4, 1 + w, 8 * j + 1);
        uint32_t sc[32];
        tmem_ld32(s_addr, sc);
        tmem_wait_ld();
        const int y0 = j * kBN + 32 * cq;
        if (j * kBN + kBN - 1 > it.x0[w]) {  // the tile reaches past the first row's position: causal mask
#pragma unroll
          for (int i = 0; i < 32; ++i)
            if (y0 + i > x) sc[i] = 0xff800000u;  // -inf
        }
        float mx0 = -INFINITY, mx1 = -INFINITY;
#pragma unroll
        for (int i = 0; i < 16; ++i) {
          mx0 = fmaxf(mx0, __uint_as_float(sc[i]));
          mx1 = fmaxf(mx1, __uint_as_float(sc[16 + i]));
        }
        // row maximum = max over the four column quarters, exchanged through shared memory.  The exchange is
        // asynchronous (an mbarrier, one arrival per warp of the quarter): the exponentials are computed at once
        // against the row's CURRENT reference m and kept in registers; by the time they are done the other
        // quarters' maxima are there, and only if the row's maximum tops m by more than 2^8 (rare) are O and l
        // rescaled and the exponentials redone.  The first tile of an item has no reference yet and waits.
        PFD(n_done == kTraceItem && warp == 4, 1 + w, 8 * j + 2);
        float(*mxq)[kBM] = s.mxch[n_x & 1];
        mxq[cq][row] = fmaxf(mx0, mx1);
        __syncwarp();
        if (lane == 0) mbar_arrive(&s.xch[q4]);
        const uint32_t xph = n_x & 1u;
        ++n_x;
        auto row_max = [&]() {
          mbar_wait(&s.xch[q4], xph);
          return fmaxf(fmaxf(mxq[0][row], mxq[1][row]), fmaxf(mxq[2][row], mxq[3][row]));
        };
        uint32_t pk[16];
        auto exponentials = [&](float mref, unsigned long long lin) {
          // P = exp2(c2 s - c2 m) as bf16 pairs; returns l + their sum
          const float ms = -mref * c2;
          const unsigned long long msp = pack2f(ms, ms);
#pragma unroll
          for (int i = 0; i < 16; ++i) {
            const unsigned long long e2 = ffma2(pack2f(__uint_as_float(sc[2 * i]), __uint_as_float(sc[2 * i + 1])), c2p, msp);
            float p0, p1;
            if ((i & 7) < kEmuOf8) {
              const unsigned long long pp = ex2_fma2(e2);
              unpack2f(pp, p0, p1);
              lin = fadd2(lin, pp);
            } else {
              float e0, e1;
              unpack2f(e2, e0, e1);
              p0 = ex2(e0), p1 = ex2(e1);
              lin = fadd2(lin, pack2f(p0, p1));
            }
            pk[i] = pack_bf16(p0, p1);
          }
          return lin;
        };
        if (j == 0) {
          m = row_max();  // key 0 <= every query position: finite
          l2 = exponentials(m, l2);
        } else {
          const unsigned long long l_try = exponentials(m, l2);
          PFD(n_done == kTraceItem && warp == 4, 1 + w, 8 * j + 3);
          const float m_new = fmaxf(m, row_max());
          const bool need = (m_new - m) * c2 > kRescaleLog2;   // same decision in all four warps of the row
          if (__any_sync(0xffffffffu, need)) {
            // rescale (this thread's quarter of) O and l of the rows whose reference maximum moves; PV(w, j-1) has
            // landed: S(w, j) was issued behind it
            const float f = need ? ex2((m - m_new) * c2) : 1.f;
            uint32_t o[32];
            tmem_ld32(o_addr, o);
            tmem_wait_ld();
#pragma unroll
            for (int i = 0; i < 32; ++i) o[i] = __float_as_uint(__uint_as_float(o[i]) * f);
            tmem_st32(o_addr, o);
            float la, lb;
            unpack2f(l2, la, lb);
            if (need) m = m_new;
            l2 = exponentials(m, pack2f(la * f, lb * f));
          } else {
            l2 = l_try;
          }
        }
        // P goes over the first 16 of this thread's OWN 32 score columns (keys 32 cq .. at columns 32 cq ..): no
        // thread writes what another still reads
        PFD(n_done == kTraceItem && warp == 4, 1 + w, 8 * j + 4);
        tmem_st16(s_addr, pk);
        tmem_wait_st();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(&s.p_ready[w]);
        PFD(n_done == kTraceItem && warp == 4, 1 + w, 8 * j + 5);
      };
      auto hand_over = [&](auto wc) {
        // the row block's partial row sums and reference maxima go to the epilogue warps; this warp moves on
        constexpr int w = decltype(wc)::value;
        if (it.nkt[w] == 0) return;
        const uint32_t par = n_fin[w] & 1u;
        // not before the epilogue has taken the previous item's: an item of a single tile needs no PV - no o_free - to
        // get here, and l_ready must never run two phases ahead of its waiter (a parity wait could not tell)
        mbar_wait(&s.l_free[w], par ^ 1u);
        ++n_fin[w];
        float la, lb;
        unpack2f(l_[w], la, lb);
        s.lfin[par][w][cq][row] = la + lb;
        if (cq == 0) s.mfin[par][w][row] = m_[w];
        __syncwarp();
        if (lane == 0) mbar_arrive(&s.l_ready[w]);
      };
      constexpr std::integral_constant<int, 0> W0{};
      constexpr std::integral_constant<int, 1> W1{};
      if (warp == 4) PFT(1, 8 * n_done + 0);
      for (int j = 0; j < it.n_kt; ++j) {
        if (j < it.nkt[0]) tile(W0, j);
        if (j < it.nkt[1]) tile(W1, j);
      }
      if (warp == 4) PFT(1, 8 * n_done + 1);
      hand_over(W0);
      hand_over(W1);
      if (warp == 4) PFT(1, 8 * n_done + 2);
      ++n_done;
    }
  } else {
    // ============================== epilogue warps ==============================
    // One warp per tensor-memory lane quarter: O_w / l -> bf16 -> out for the quarter's 32 rows, off the softmax
    // warps' path (they are already on the next item's first tiles).  out rows are 7 KB apart - 32 lanes storing 16
    // bytes each would touch 32 lines per instruction - so a warp stages [32 rows][64 bf16] of one d-half in shared
    // memory (128-byte swizzle) and one TMA store writes it as 32 full 128-byte row segments; rows past the end of
    // the call's range are clipped by the tensor map.
    set_regs_dec<kRegsEpilogue>();
    const int q4 = warp & 3;
    const int row = q4 * 32 + lane;
    const uint32_t lane_base = tb + ((uint32_t)(q4 * 32) << 16);
    uint8_t* stage = s.ostage[q4];
    uint32_t n_pv[2] = {0u, 0u}, n_fin[2] = {0u, 0u};
    for (int id = first; id < n_items; id += stride) {
      const Item it = make_item(id, c, prm, len);
#pragma unroll
      for (int w = 0; w < 2; ++w) {
        if (it.nkt[w] == 0) continue;
        n_pv[w] += (uint32_t)it.nkt[w];
        const uint32_t par = n_fin[w] & 1u;
        ++n_fin[w];
        mbar_wait(&s.l_ready[w], par);
        const float l = (s.lfin[par][w][0][row] + s.lfin[par][w][1][row]) + (s.lfin[par][w][2][row] + s.lfin[par][w][3][row]);
        const float m = s.mfin[par][w][row];
        __syncwarp();
        if (lane == 0) mbar_arrive(&s.l_free[w]);
        mbar_wait(&s.o_done[w], (n_pv[w] - 1u) & 1u);   // the item's last PV of this row block
        tc_fence_after();
        const float inv = 1.f / l;
        const int x = it.x0[w] + row;
#pragma unroll
        for (int h = 0; h < 2; ++h) {
#pragma unroll
          for (int cc = 0; cc < 2; ++cc) {
            uint32_t o[32];
            tmem_ld32(lane_base + 256u + 128u * w + 64u * h + 32u * cc, o);
            tmem_wait_ld();
            if (h == 1 && cc == 1) {  // O_w is in registers / on its way out: the next item may overwrite it
              tc_fence_before();
              __syncwarp();
              if (lane == 0) mbar_arrive(&s.o_free[w]);
            }
#pragma unroll
            for (int v4 = 0; v4 < 4; ++v4) {
              uint4 val;
              val.x = pack_bf16(__uint_as_float(o[8 * v4 + 0]) * inv, __uint_as_float(o[8 * v4 + 1]) * inv);
              val.y = pack_bf16(__uint_as_float(o[8 * v4 + 2]) * inv, __uint_as_float(o[8 * v4 + 3]) * inv);
              val.z = pack_bf16(__uint_as_float(o[8 * v4 + 4]) * inv, __uint_as_float(o[8 * v4 + 5]) * inv);
              val.w = pack_bf16(__uint_as_float(o[8 * v4 + 6]) * inv, __uint_as_float(o[8 * v4 + 7]) * inv);
              *reinterpret_cast<uint4*>(stage + lane * 128 + (((cc * 4 + v4) ^ (lane & 7)) << 4)) = val;
            }
          }
          asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
          __syncwarp();
          if (lane == 0) {
            tma_store_4d(&tm_o, stage, 64 * h, it.hq[w], it.x0[w] - prm.pos_begin + 32 * q4, it.lc);
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
            asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");   // the staging slice has been read
          }
          __syncwarp();
        }
        if (x <= it.xl[w] && prm.lse != nullptr) {
          const size_t orow = ((size_t)it.lc * prm.n_tok + (size_t)(x - prm.pos_begin)) * c.n_q + it.hq[w];
          prm.lse[orow] = m * prm.sm_scale + __logf(l);
        }
      }
    }
  }
  // ---- teardown: the single-lane roles diverged - reconverge before the aligned CTA barrier ----------
  __syncwarp();
  tc_fence_before();
  __syncthreads();
  if (warp == 1) tmem_dealloc(0u, kTmemCols);
}

}  // namespace

cudaError_t launch_prefill_attn_umma(const CacheView& c, int seq, int pos_begin, int n_tok, const void* q, void* out,
                                     float* lse, int layer_begin, int layer_end, float sm_scale, int sm_count,
                                     cudaStream_t st, LaunchInfo* info) {
  const int n_layers_call = layer_end - layer_begin;
  CUtensorMap tm_q, tm_k, tm_v, tm_o;
  {
    const uint64_t dims[4] = {128, (uint64_t)c.n_q, (uint64_t)n_tok, (uint64_t)n_layers_call};
    const uint64_t str[3] = {256, (uint64_t)c.n_q * 256, (uint64_t)n_tok * c.n_q * 256};
    const uint32_t box[4] = {64, 1, (uint32_t)kBM, 1};
    if (!encode_tmap_bf16(&tm_q, q, 4, dims, str, box, true)) return cudaErrorInvalidValue;
    const uint32_t obox[4] = {64, 1, 32, 1};  // one lane quarter's rows of one d-half
    if (!encode_tmap_bf16(&tm_o, out, 4, dims, str, obox, true)) return cudaErrorInvalidValue;
  }
  {
    const uint64_t dims[5] = {128, (uint64_t)c.p, (uint64_t)c.n_kv, (uint64_t)c.n_pages, (uint64_t)c.n_layers};
    const uint64_t str[4] = {256, (uint64_t)c.p * 256, (uint64_t)c.n_kv * c.p * 256, (uint64_t)c.n_pages * c.n_kv * c.p * 256};
    const uint32_t box[5] = {64, (uint32_t)c.p, 1, 1, 1};
    if (!encode_tmap_bf16(&tm_k, c.k_pool, 5, dims, str, box, false)) return cudaErrorInvalidValue;
    if (!encode_tmap_bf16(&tm_v, c.v_pool, 5, dims, str, box, false)) return cudaErrorInvalidValue;
  }
  const int smem = (int)sizeof(USmem) + 1024;  // + slack for the 1024-byte alignment of the tiles
  cudaError_t ea = opt_in_smem_once(kSmemPrefillUmma, reinterpret_cast<const void*>(prefill_umma_kernel), smem);
  if (ea != cudaSuccess) return ea;
  UParams prm{};
  prm.out = reinterpret_cast<uint16_t*>(out);
  prm.lse = lse;
  prm.seq = seq;
  prm.pos_begin = pos_begin;
  prm.n_tok = n_tok;
  prm.layer_begin = layer_begin;
  prm.sm_scale = sm_scale;
  const int n_qb = (n_tok + kBM - 1) / kBM;
  const int n_pairs = (n_qb * c.group + 1) / 2;
  const int n_items = n_pairs * c.n_kv * n_layers_call;
  const int grid = n_items < sm_count ? n_items : sm_count;  // persistent: one CTA per SM
  prefill_umma_kernel<<<grid, kUThreads, smem, st>>>(tm_q, tm_k, tm_v, tm_o, c, prm, n_items);
  info->launches += 1;
  info->grid = grid;
  info->smem = smem;
  return cudaGetLastError();
}

}  // namespace murmur

#ifdef MURMUR_PFTRACE
extern "C" __attribute__((visibility("default"))) int murmur_debug_pftrace(long long* host_out) {
  cudaDeviceSynchronize();
  return (int)cudaMemcpyFromSymbol(host_out, murmur::g_pftrace, sizeof(long long) * 2 * 8192);
}
extern "C" __attribute__((visibility("default"))) int murmur_debug_pftile(long long* host_out) {
  cudaDeviceSynchronize();
  return (int)cudaMemcpyFromSymbol(host_out, murmur::g_pftile, sizeof(long long) * 3 * 1024);
}
#endif
