// S6, CTA-pair variant: tensor-core patch attention with tcgen05 cta_group::2 (cache-patching, Eq. 6, PAPER.md:118-123,
// 718).  For tasks with more than 128 query rows per kv head and head_dim 128.
//
// Why pairs.  With two Q tiles in ONE CTA (fcg_attn_tc.cu, <2,1>) every 64-token step moves 160 KB through the SM's
// shared-memory port (Q is re-read for every KV tile: 64 KB, K 32 KB, V 32 KB, TMA writes 32 KB) = 1250 cycles of a
// 128 B/clk port against 1024 cycles of MMA: the port, not the tensor pipe, paces the kernel (ncu: port 67 %, tensor pipe
// 68 % on C5, 56 % on C4's 129..256-row class).  A CTA pair on the two SMs of a TPC holds ONE Q tile per SM and splits
// every K/V tile between the two shared memories (tcgen05.mma.cta_group::2: each SM feeds its half of the B operand
// to both tensor cores): per 128-token step and SM the port moves Q 32 KB + K 16 KB + V 16 KB + TMA writes 32 KB =
// 96 KB = 768 cycles against the same 1024 cycles of MMA, and each SM pulls only half of the K/V bytes.
//
//   cluster = 2 CTAs = (KV split x row group of 256 rows, kv head, layer x task); CTA r of the pair owns query rows
//             [r*128, r*128 + 128) of the group: its Q tile, its softmax warps, its S / P / O in its own TMEM.
//   KV tile = 128 tokens.  S = Q K^T: M = 256 (128 per CTA), N = 128, K = 128; the B operand K is N-split: CTA r holds the
//             tile's tokens [r*64, r*64 + 64) (both 64-column halves).  O += P V: M = 256, N = 128 (head_dim), K = 128
//             tokens; A = P from each CTA's TMEM; the B operand V is N-split: CTA r holds columns [r*64, r*64 + 64) of
//             all 128 tokens.
//   warps   = 8 softmax warps, K loader, V loader, MMA warp.  Softmax warp w serves the TMEM lane quarter w % 4 (32 query
//             rows) and the column half w / 4 of every S tile: two warps per SM sub-partition hide each other's TMEM /
//             MUFU latencies (with one, the softmax chain paced the kernel at half speed); the two threads of a row
//             exchange their partial row maxima through shared memory (one 64-thread named barrier per tile) and
//             split the O rescale and the epilogue by columns.  The MMA warp of the leader CTA (rank 0) issues every
//             tcgen05.mma of the pair, the other one only allocates / frees TMEM.
//   TMEM    = 512 columns per CTA: S[b] at b*128, O at 256, P[b] at 384 + b*64.
//   barriers: the TMA loads of BOTH CTAs complete on the leader's k_full / v_full (cta_group::2 form, leader arms the
//             expected bytes of the pair); s_free / p_full / q_ready live in the leader and count one arrival per
//             softmax warp of the pair (16; remote mbarrier.arrive from rank 1); k_empty / v_empty / s_full / pv_done /
//             all_done are signalled in both CTAs at once by tcgen05.commit ... multicast::cluster.
//   Tail    : the V rows of the last tile that hold no token of the split are zeroed in shared memory before P V (0 x NaN):
//             for that tile each V loader lands its half on a barrier of its own CTA, zeroes, and then arrives on v_full.
//   Output  : final bf16 rows (one split) or fp32 (m, l, o) partials for attn_combine_kernel, as in fcg_attn_tc.cu.
#include <cuda_bf16.h>

#include "fcg_internal.h"
#include "fcg_tc_common.cuh"

namespace fcg {
namespace {

constexpr int PBM = 128;        // query rows per CTA
constexpr int PBN = 128;        // cache tokens per pair tile
constexpr int PD = 128;         // head_dim
constexpr float P_RESCALE_TAU = 8.0f;

// ---- cluster helpers ------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t cluster_ctarank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
  return r;
}
__device__ __forceinline__ void cluster_sync_all() {
  asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
  asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// shared::cluster address of `local` (a shared::cta address of this CTA) in CTA `rank` of the cluster
__device__ __forceinline__ uint32_t map_to_rank(uint32_t local, uint32_t rank) {
  uint32_t r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(local), "r"(rank));
  return r;
}
// Arrivals on a barrier of the leader CTA.  The hot ones (S read, P written: twice per tile and warp) order tcgen05
// traffic only, which tcgen05.fence::before_thread_sync already does: the default (.release.cta) form.  A cluster-scope
// release costs a full memory barrier per arrival -- the first version of this kernel spent most of its stall samples
// there (ncu: stalled_membar) and ran at half the speed of the single-CTA kernel.  The two arrivals that publish
// generic-proxy shared-memory writes (Q tile, zeroed V rows) keep the cluster-scope release; they run once per CTA.
__device__ __forceinline__ void mbar_arrive_cluster(uint32_t cluster_addr) {
  asm volatile("mbarrier.arrive.shared::cluster.b64 _, [%0];" ::"r"(cluster_addr) : "memory");
}
__device__ __forceinline__ void mbar_arrive_cluster_release(uint32_t cluster_addr) {
  asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" ::"r"(cluster_addr) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait_cluster(uint32_t bar, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%1], %2;\n\t"
      "selp.u32 %0, 1, 0, p;\n\t"
      "}"
      : "=r"(ok)
      : "r"(bar), "r"(parity)
      : "memory");
  return ok != 0;
}
__device__ __forceinline__ void mbar_wait_cluster(uint32_t bar, uint32_t parity) {
  while (!mbar_try_wait_cluster(bar, parity)) {
  }
}

// ---- cta_group::2 forms -----------------------------------------------------------------------------
__device__ __forceinline__ void tmem_alloc_pair(uint32_t smem_dst) {
  asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_dst) : "memory");
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc_pair(uint32_t taddr) {
  asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, 512;" ::"r"(taddr) : "memory");
}
// arrive on the barrier at this shared-memory offset in BOTH CTAs once every tcgen05.mma issued so far has completed
__device__ __forceinline__ void umma_commit_pair(uint32_t bar) {
  if (elect_one())
  asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;" ::"r"(bar),
               "h"((unsigned short)3)
               : "memory");
}
__device__ __forceinline__ void umma_ss_pair(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
  if (elect_one())
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, p;\n\t"
      "}" ::"r"(d_tmem),
      "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate)
      : "memory");
}
__device__ __forceinline__ void umma_ts_pair(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
  if (elect_one())
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::2.kind::f16 [%0], [%1], %2, %3, p;\n\t"
      "}" ::"r"(d_tmem),
      "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(accumulate)
      : "memory");
}
// TMA box whose completion bytes go to a barrier of the pair's leader CTA (`bar_cluster`: a shared::cluster address)
__device__ __forceinline__ void tma_load_5d_pair(uint32_t dst, const TmaDesc *desc, uint32_t bar_cluster, int c0, int c1, int c2, int c3,
                                                 int c4) {
  if (elect_one())
  asm volatile(
      "cp.async.bulk.tensor.5d.cta_group::2.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5, %6}], [%7];" ::"r"(
          dst),
      "l"(reinterpret_cast<uint64_t>(desc)), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4), "r"(bar_cluster)
      : "memory");
}

// ---- shared memory map (per CTA; identical offsets in both CTAs of the pair) -------------------------
struct PC {
  static constexpr int SK = 6, SV = 5;     // 128-token steps: 6 x 16 KB of K, 5 x 16 KB of V per CTA (227 KB limit)
  static constexpr int Q_B = PBM * PD * 2;              // 32 KB: two 64-column halves of [128][128 B]
  static constexpr int K_B = (PBN / 2) * PD * 2;        // 16 KB: this CTA's 64 tokens, two halves of [64][128 B]
  static constexpr int V_B = PBN * (PD / 2) * 2;        // 16 KB: all 128 tokens x this CTA's 64 columns, [128][128 B]
  static constexpr int OFF_Q = 0, OFF_K = OFF_Q + Q_B, OFF_V = OFF_K + SK * K_B, OFF_BAR = OFF_V + SV * V_B;
  // k_full[SK] k_empty[SK] v_full[SV] v_empty[SV] v_land[SV] s_full[2] s_free[2] p_full[2] pv_done[2] q_ready all_done
  static constexpr int N_BARS = 2 * SK + 3 * SV + 8 + 2;
  static constexpr int OFF_X = OFF_BAR + N_BARS * 8 + 16;          // float xch[2][2][128]: partial row maxima / sums
  static constexpr int SMEM_BYTES = OFF_X + 2 * 2 * 128 * 4 + 1024;
  static constexpr int N_SOFTMAX = 256;
  static constexpr int NTHREADS = N_SOFTMAX + 96;
  static constexpr int KLOAD_WARP = 8, VLOAD_WARP = 9, MMA_WARP = 10;
  static constexpr int TM_S = 0, TM_O = 256, TM_P = 384;
};

__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(PC::NTHREADS, 1)
    attn_pair_kernel(const AttnParams p, const __grid_constant__ TmaDesc tm_k, const __grid_constant__ TmaDesc tm_v) {
  constexpr int SK = PC::SK, SV = PC::SV;
  extern __shared__ unsigned char smem_raw[];
  unsigned char *smem = reinterpret_cast<unsigned char *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  const uint32_t sbase = smem_u32(smem);
  const uint32_t rank = cluster_ctarank();
  const bool leader = rank == 0;

  const int task_i = blockIdx.z % p.n_tasks;
  const int li = blockIdx.z / p.n_tasks;
  const AttnTaskDev tk = p.tasks[task_i];
  const int pair_x = blockIdx.x >> 1;
  const int split = pair_x % p.max_splits;
  const int rg = pair_x / p.max_splits;
  const int G = p.group;
  const int R = tk.n * G;
  const int row0 = rg * (2 * PBM);                // first query row of the pair
  // (both CTAs of a pair take the same decision: no half-exited cluster)
  if (split >= tk.n_splits || row0 >= R) return;
  const int g = blockIdx.y;
  const int layer = p.layer_begin + li;
  const int tid = threadIdx.x, lane = tid & 31;
  const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);

  const int Rp = min(R - row0, 2 * PBM);          // valid query rows of the pair
  const int my_rows = max(0, min(Rp - (int)rank * PBM, PBM));   // valid rows of this CTA's Q tile (may be 0 for rank 1)
  const int t_begin = split * tk.split_len;
  const int t_end = min(tk.kv_len, t_begin + tk.split_len);
  const int32_t *pos = p.positions + tk.tok_off;
  const int pair_max_lim = min(pos[(row0 + Rp - 1) / G], t_end - 1);
  const int n_tiles = pair_max_lim >= t_begin ? (pair_max_lim - t_begin) / PBN + 1 : 0;

  const uint32_t bar0 = sbase + PC::OFF_BAR;
  auto k_full = [&](int s) { return bar0 + 8 * s; };
  auto k_empty = [&](int s) { return bar0 + 8 * (SK + s); };
  auto v_full = [&](int s) { return bar0 + 8 * (2 * SK + s); };
  auto v_empty = [&](int s) { return bar0 + 8 * (2 * SK + SV + s); };
  auto v_land = [&](int s) { return bar0 + 8 * (2 * SK + 2 * SV + s); };
  constexpr int B0 = 2 * SK + 3 * SV;
  auto s_full = [&](int b) { return bar0 + 8 * (B0 + b); };
  auto s_free = [&](int b) { return bar0 + 8 * (B0 + 2 + b); };
  auto p_full = [&](int b) { return bar0 + 8 * (B0 + 4 + b); };
  auto pv_done = [&](int b) { return bar0 + 8 * (B0 + 6 + b); };
  const uint32_t q_ready = bar0 + 8 * (B0 + 8);
  const uint32_t all_done = bar0 + 8 * (B0 + 9);
  const uint32_t tmem_slot = bar0 + 8 * PC::N_BARS;
  volatile uint32_t *tmem_slot_ptr = reinterpret_cast<volatile uint32_t *>(smem + PC::OFF_BAR + 8 * PC::N_BARS);

  if (tid == 0) {
    for (int s = 0; s < SK; ++s) {
      mbar_init(k_full(s), 1);                     // leader: its K loader's arrive.expect_tx (bytes of the pair)
      mbar_init(k_empty(s), 1);                    // multicast commit
    }
    for (int s = 0; s < SV; ++s) {
      mbar_init(v_full(s), 3);                     // leader: its V loader's arrive.expect_tx + one arrival per V loader of the pair
      mbar_init(v_empty(s), 1);
      mbar_init(v_land(s), 1);                     // own CTA: the ragged last tile lands here first
    }
    for (int b = 0; b < 2; ++b) {
      mbar_init(s_full(b), 1);                     // multicast commit
      mbar_init(s_free(b), 16);                    // leader: one arrival per softmax warp of the pair
      mbar_init(p_full(b), 16);
      mbar_init(pv_done(b), 1);
    }
    mbar_init(q_ready, 16);
    mbar_init(all_done, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == PC::KLOAD_WARP && lane == 0) tma_prefetch_desc(&tm_k);
  if (warp == PC::VLOAD_WARP && lane == 0) tma_prefetch_desc(&tm_v);
  __syncthreads();
  // both CTAs' barriers exist before anybody signals across the pair, and the pair allocates TMEM together
  cluster_sync_all();
  if (warp == PC::MMA_WARP) tmem_alloc_pair(tmem_slot);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = __shfl_sync(0xffffffffu, *tmem_slot_ptr, 0);
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");

  // leader-side barriers as seen from this CTA
  auto on_leader = [&](uint32_t local) { return map_to_rank(local, 0); };

  if (warp == PC::KLOAD_WARP) {
    // ======================================= K loader =======================================
    // this CTA's 64 tokens of every 128-token tile: pages through the page table, two box copies per page
    const int P = p.page_size;
    const int pshift = __ffs(P) - 1;
    const int pph = (PBN / 2) >> pshift;            // pages per 64-token half tile
    const int32_t *table = p.tables + tk.table_off + (t_begin >> pshift);
    const int n_pages_split = (t_end - t_begin + P - 1) >> pshift;
    auto page_of = [&](int j) -> int {
      const int pi = (2 * j + (int)rank) * pph + lane;
      return (lane < pph && pi < n_pages_split) ? __ldg(table + pi) : -1;
    };
    auto n_ok_of = [&](int j, int r) { return max(0, min(pph, n_pages_split - (2 * j + r) * pph)); };
    int page = page_of(0);
    int st = 0, round = 0;
    for (int j = 0; j < n_tiles; ++j) {
      const int page_next = page_of(j + 1);
      if (round > 0) mbar_wait(k_empty(st), (round - 1) & 1);
      const int n_ok = n_ok_of(j, (int)rank);
      const uint32_t dst = sbase + PC::OFF_K + st * PC::K_B;
      const uint32_t bar = on_leader(k_full(st));
      if (leader && elect_one()) mbar_arrive_expect_tx(k_full(st), (uint32_t)((n_ok_of(j, 0) + n_ok_of(j, 1)) * P * (PD * 2)));
#pragma unroll 1
      for (int i = 0; i < n_ok; ++i) {
        const int pg = __shfl_sync(0xffffffffu, page, i);
        tma_load_5d_pair(dst + i * P * 128, &tm_k, bar, 0, 0, g, pg, layer);
        tma_load_5d_pair(dst + i * P * 128 + (PBN / 2) * 128, &tm_k, bar, 64, 0, g, pg, layer);
      }
      page = page_next;
      if (++st == SK) {
        st = 0;
        ++round;
      }
    }
  } else if (warp == PC::VLOAD_WARP) {
    // ======================================= V loader =======================================
    // all 128 tokens of every tile, this CTA's 64 columns: one box copy per page
    const int P = p.page_size;
    const int pshift = __ffs(P) - 1;
    const int ppt = PBN >> pshift;                  // pages per tile (P = 8: 16 pages; lanes 0..15)
    const int32_t *table = p.tables + tk.table_off + (t_begin >> pshift);
    const int n_pages_split = (t_end - t_begin + P - 1) >> pshift;
    auto page_of = [&](int j) -> int {
      const int pi = j * ppt + lane;
      return (lane < ppt && pi < n_pages_split) ? __ldg(table + pi) : -1;
    };
    int page = page_of(0);
    int st = 0, round = 0;
    const uint32_t me_on_leader = 0;
    (void)me_on_leader;
    for (int j = 0; j < n_tiles; ++j) {
      const int page_next = page_of(j + 1);
      if (round > 0) mbar_wait(v_empty(st), (round - 1) & 1);
      const int n_ok = min(ppt, n_pages_split - j * ppt);
      const uint32_t dst = sbase + PC::OFF_V + st * PC::V_B;
      const int ts = t_begin + j * PBN;
      const bool ragged = ts + PBN > t_end;           // only the last tile of the split
      const uint32_t bytes = (uint32_t)(n_ok * P * 128);
      if (!ragged) {
        const uint32_t bar = on_leader(v_full(st));
        if (leader && elect_one()) mbar_arrive_expect_tx(v_full(st), 2 * bytes);
#pragma unroll 1
        for (int i = 0; i < n_ok; ++i) {
          const int pg = __shfl_sync(0xffffffffu, page, i);
          tma_load_5d_pair(dst + i * P * 128, &tm_v, bar, 64 * (int)rank, 0, g, pg, layer);
        }
        if (elect_one()) mbar_arrive_cluster(bar);
      } else {
        // land on a barrier of this CTA, zero the rows that hold no token of the split, then report to the leader
        if (elect_one()) mbar_arrive_expect_tx(v_land(st), bytes);
#pragma unroll 1
        for (int i = 0; i < n_ok; ++i) {
          const int pg = __shfl_sync(0xffffffffu, page, i);
          tma_load_5d(dst + i * P * 128, &tm_v, v_land(st), 64 * (int)rank, 0, g, pg, layer);
        }
        mbar_wait(v_land(st), 0);                     // used once per CTA (one ragged tile per split)
        const int r0 = t_end - ts;
        unsigned char *vt = smem + PC::OFF_V + st * PC::V_B;
        for (int i = lane; i < (PBN - r0) * 8; i += 32) {
          const int row = r0 + (i >> 3), c = i & 7;
          *reinterpret_cast<uint4 *>(vt + row * 128 + (c << 4)) = make_uint4(0, 0, 0, 0);
        }
        fence_proxy_async();
        __syncwarp();
        if (leader && elect_one()) mbar_arrive(v_full(st));           // the leader's own "expect" arrival (no bytes)
        if (elect_one()) mbar_arrive_cluster_release(on_leader(v_full(st)));
      }
      page = page_next;
      if (++st == SV) {
        st = 0;
        ++round;
      }
    }
  } else if (warp == PC::MMA_WARP) {
    // ======================================= MMA issuer (leader only) ===========================
    if (leader && n_tiles > 0) {
      constexpr uint32_t IDESC_S = idesc_f16(PBN, false, 256);
      constexpr uint32_t IDESC_O = idesc_f16(PD, true, 256);
      mbar_wait_cluster(q_ready, 0);
      const uint64_t qdesc0 = smem_desc(sbase + PC::OFF_Q, 16, 1024);
      const uint64_t kdesc0 = smem_desc(sbase + PC::OFF_K, 16, 1024);
      const uint64_t vdesc0 = smem_desc(sbase + PC::OFF_V, PBN * 128, 1024);   // MN-major; one 64-column atom per CTA
      int sk = 0, rk = 0;
      auto issue_qk = [&](int j) {
        if (j >= 2) mbar_wait(s_free(j & 1), ((j - 2) >> 1) & 1);   // both CTAs have read S[j&1] of tile j-2
        mbar_wait(k_full(sk), rk & 1);
        const uint64_t kdesc = kdesc0 + (uint64_t)((sk * PC::K_B) >> 4);
        tc_fence_after();
#pragma unroll
        for (int k = 0; k < PD / 16; ++k) {
          const uint64_t a = qdesc0 + (uint64_t)(((k >> 2) * (PBM * 128) + (k & 3) * 32) >> 4);
          const uint64_t b = kdesc + (uint64_t)(((k >> 2) * ((PBN / 2) * 128) + (k & 3) * 32) >> 4);
          umma_ss_pair(tmem_base + PC::TM_S + (j & 1) * PBN, a, b, IDESC_S, k > 0);
        }
        umma_commit_pair(s_full(j & 1));
        umma_commit_pair(k_empty(sk));
        if (++sk == SK) {
          sk = 0;
          ++rk;
        }
      };
      int sv = 0, rv = 0;
      auto issue_pv = [&](int j) {
        mbar_wait_cluster(v_full(sv), rv & 1);
        mbar_wait(p_full(j & 1), (j >> 1) & 1);
        tc_fence_after();
        const uint64_t vdesc = vdesc0 + (uint64_t)((sv * PC::V_B) >> 4);
        const uint32_t tmem_p = tmem_base + PC::TM_P + (j & 1) * (PBN / 2);
#pragma unroll
        for (int k = 0; k < PBN / 16; ++k)
          umma_ts_pair(tmem_base + PC::TM_O, tmem_p + k * 8, vdesc + (uint64_t)((k * 2048) >> 4), IDESC_O, (j > 0 || k > 0) ? 1u : 0u);
        umma_commit_pair(v_empty(sv));
        umma_commit_pair(pv_done(j & 1));
        if (++sv == SV) {
          sv = 0;
          ++rv;
        }
      };
      issue_qk(0);
      if (n_tiles > 1) issue_qk(1);
      for (int j = 0; j < n_tiles; ++j) {
        if (j + 2 < n_tiles) issue_qk(j + 2);
        issue_pv(j);
      }
      umma_commit_pair(all_done);
    }
  } else {
    // ======================================= softmax ========================================
    // this CTA's Q tile: MMA row m holds query row row0 + rank*128 + m; rows past the valid ones are zero
    {
      uint4 qv[8];
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        const int ci = tid + PC::N_SOFTMAX * i;
        const int row = ci >> 4, c = ci & 15;
        qv[i] = make_uint4(0, 0, 0, 0);
        if (row < my_rows) {
          const int r = row0 + (int)rank * PBM + row;
          const uint16_t *src = p.q + (((size_t)li * p.n_total + tk.tok_off + r / G) * p.n_q_heads + g * G + r % G) * PD + c * 8;
          qv[i] = __ldg(reinterpret_cast<const uint4 *>(src));
        }
      }
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        const int ci = tid + PC::N_SOFTMAX * i;
        const int row = ci >> 4, c = ci & 15;
        const uint32_t dst = PC::OFF_Q + (c >> 3) * (PBM * 128) + row * 128 + (((c & 7) ^ (row & 7)) << 4);
        *reinterpret_cast<uint4 *>(smem + dst) = qv[i];
      }
    }
    fence_proxy_async();
    __syncwarp();
    if (lane == 0) mbar_arrive_cluster_release(on_leader(q_ready));

    const int quarter = warp & 3, half = warp >> 2;      // TMEM lane quarter (rows), column half of every S tile
    const int row = quarter * 32 + lane;                 // 0..127 == TMEM lane
    const uint32_t lane_addr = ((uint32_t)(quarter * 32) << 16);
    const int r = row0 + (int)rank * PBM + row;
    const bool valid = row < my_rows;
    const int lim = valid ? min(pos[r / G], t_end - 1) : -1;
    const uint32_t tmem_s = tmem_base + lane_addr + PC::TM_S + half * 64;
    const uint32_t tmem_o = tmem_base + lane_addr + PC::TM_O + half * 64;
    const uint32_t tmem_p = tmem_base + lane_addr + PC::TM_P + half * 32;
    const uint32_t s_free_l0 = on_leader(s_free(0)), p_full_l0 = on_leader(p_full(0));
    float *xch = reinterpret_cast<float *>(smem + PC::OFF_X);          // [parity][half][row]
    const float sc = p.scale_log2;
    float m_ref = -INFINITY;
    float l = 0.f;
    // the two warps that share this lane quarter meet at a named barrier of their own (ids 1..4, 64 threads)
    auto pair_sync = [&]() { asm volatile("bar.sync %0, 64;" ::"r"(quarter + 1) : "memory"); };

    for (int j = 0; j < n_tiles; ++j) {
      const int ts = t_begin + j * PBN + half * 64;      // token of this thread's first column
      const int b = j & 1;
      mbar_wait(s_full(b), (j >> 1) & 1);
      tc_fence_after();
      uint32_t sreg[64];
      TMEM_LD_32(tmem_s + b * PBN, sreg);
      TMEM_LD_32(tmem_s + b * PBN + 32, (sreg + 32));
      tmem_wait_ld();
      // S[b] is in registers: Q K^T of tile j+2 may overwrite it
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive_cluster(s_free_l0 + 8 * b);
      if (ts + 63 > lim) {
#pragma unroll
        for (int c = 0; c < 64; ++c)
          if (ts + c > lim) sreg[c] = 0xff800000u;       // -inf, by selection (S may be garbage there)
      }
      float mx4[4] = {-INFINITY, -INFINITY, -INFINITY, -INFINITY};
#pragma unroll
      for (int c = 0; c < 64; ++c) mx4[c & 3] = fmaxf(mx4[c & 3], __uint_as_float(sreg[c]));
      // the row maximum needs the other column half too: the two threads of a row exchange their partial maxima through
      // shared memory (one 64-thread named barrier per tile).  Reading the other half from TMEM instead (no barrier, so
      // the two warps of a sub-partition do not run in lockstep) was measured no faster on C3 / C5 and slower on C4
      // (3.93 vs 3.62 ms): the extra 64 max operations cost what the lockstep does.
      float mx = fmaxf(fmaxf(mx4[0], mx4[1]), fmaxf(mx4[2], mx4[3]));
      xch[(b * 2 + half) * 128 + row] = mx;
      pair_sync();
      mx = fmaxf(mx, xch[(b * 2 + (half ^ 1)) * 128 + row]);
      const float m_new = fmaxf(m_ref, mx * sc);
      float factor = 1.f;
      const bool bump = (m_new - m_ref > P_RESCALE_TAU) || (m_ref == -INFINITY && m_new != -INFINITY);
      if (bump) {
        factor = (m_ref == -INFINITY) ? 0.f : ex2_approx(m_ref - m_new);
        m_ref = m_new;
      }
      if (j >= 1 && __any_sync(0xffffffffu, bump)) {
        mbar_wait(pv_done((j - 1) & 1), ((j - 1) >> 1) & 1);      // O holds tiles 0..j-1 once P V of tile j-1 is done
        tc_fence_after();
#pragma unroll
        for (int ch = 0; ch < 2; ++ch) {                          // this thread's half of the row's O columns
          uint32_t oreg[32];
          TMEM_LD_32(tmem_o + ch * 32, oreg);
          tmem_wait_ld();
#pragma unroll
          for (int c = 0; c < 32; ++c) oreg[c] = __float_as_uint(__uint_as_float(oreg[c]) * factor);
          TMEM_ST_32(tmem_o + ch * 32, oreg);
        }
        tmem_wait_st();
      }
      l *= factor;
      const float mu = m_ref == -INFINITY ? 0.f : m_ref;
      if (j >= 2) mbar_wait(pv_done(b), ((j - 2) >> 1) & 1);      // P[b] was last read by P V of tile j-2
      const float2 sc2 = make_float2(sc, sc), nmu2 = make_float2(-mu, -mu);
      float2 sum2[2] = {make_float2(0.f, 0.f), make_float2(0.f, 0.f)};
      uint32_t preg[32];
#pragma unroll
      for (int c8 = 0; c8 < 8; ++c8) {
        float2 e[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          const float2 x = __ffma2_rn(make_float2(__uint_as_float(sreg[c8 * 8 + 2 * q]), __uint_as_float(sreg[c8 * 8 + 2 * q + 1])), sc2, nmu2);
          e[q] = make_float2(ex2_approx(x.x), ex2_approx(x.y));
          sum2[q & 1] = __fadd2_rn(sum2[q & 1], e[q]);
        }
#pragma unroll
        for (int q = 0; q < 4; ++q) preg[c8 * 4 + q] = pack_bf16(e[q].x, e[q].y);
      }
      l += (sum2[0].x + sum2[0].y) + (sum2[1].x + sum2[1].y);
      TMEM_ST_32(tmem_p + b * (PBN / 2), preg);
      tmem_wait_st();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive_cluster(p_full_l0 + 8 * b);
    }

    // ---- epilogue: the row's two partial sums meet, then O / l -> bf16, or partials (column halves) ----------
    if (n_tiles > 0) {
      mbar_wait(all_done, 0);
      tc_fence_after();
    }
    pair_sync();                                 // the partner has read this thread's last partial maximum
    xch[half * 128 + row] = l;
    pair_sync();
    const float l_tot = l + xch[(half ^ 1) * 128 + row];
    const int i_tok = valid ? r / G : 0, hh_ = valid ? r % G : 0;
    const size_t out_row = ((size_t)li * p.n_total + tk.tok_off + i_tok) * p.n_q_heads + g * G + hh_;
    const size_t prow_i = ((size_t)(li * p.max_splits + split) * p.n_total + tk.tok_off + i_tok) * p.n_q_heads + g * G + hh_;
    const bool final_out = tk.n_splits == 1;
    const float inv = l_tot > 0.f ? 1.f / l_tot : 0.f;
#pragma unroll
    for (int ch = 0; ch < 2; ++ch) {
      uint32_t oreg[32];
      if (n_tiles > 0) {
        TMEM_LD_32(tmem_o + ch * 32, oreg);
        tmem_wait_ld();
      } else {
#pragma unroll
        for (int c = 0; c < 32; ++c) oreg[c] = 0u;
      }
      if (valid) {
        const int col0 = half * 64 + ch * 32;
        if (final_out) {
          uint16_t *dst = p.out + out_row * PD + col0;
#pragma unroll
          for (int c = 0; c < 32; c += 8) {
            uint4 v;
            v.x = pack_bf16(__uint_as_float(oreg[c]) * inv, __uint_as_float(oreg[c + 1]) * inv);
            v.y = pack_bf16(__uint_as_float(oreg[c + 2]) * inv, __uint_as_float(oreg[c + 3]) * inv);
            v.z = pack_bf16(__uint_as_float(oreg[c + 4]) * inv, __uint_as_float(oreg[c + 5]) * inv);
            v.w = pack_bf16(__uint_as_float(oreg[c + 6]) * inv, __uint_as_float(oreg[c + 7]) * inv);
            *reinterpret_cast<uint4 *>(dst + c) = v;
          }
        } else {
          float *dst = p.part_o + prow_i * PD + col0;
#pragma unroll
          for (int c = 0; c < 32; c += 4)
            *reinterpret_cast<float4 *>(dst + c) =
                make_float4(__uint_as_float(oreg[c]), __uint_as_float(oreg[c + 1]), __uint_as_float(oreg[c + 2]), __uint_as_float(oreg[c + 3]));
        }
      }
    }
    if (valid && !final_out && half == 0) *reinterpret_cast<float2 *>(p.part_ml + prow_i * 2) = make_float2(m_ref, l_tot);
  }

  // both CTAs are done with TMEM and with each other's shared memory before anything is freed
  tc_fence_before();
  __syncthreads();
  cluster_sync_all();
  if (warp == PC::MMA_WARP) {
    tc_fence_after();
    tmem_dealloc_pair(tmem_base);
  }
}

}  // namespace

// p.max_row_groups counts groups of 256 rows; grid x = 2 CTAs per (split, row group)
cudaError_t launch_attn_pair(const AttnParams &p, const TmaDesc *tm_k, const TmaDesc *tm_v, cudaStream_t stream) {
  if (!tm_k || !tm_v) return cudaErrorNotSupported;
  static bool configured[64] = {};
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess) return cudaGetLastError();
  if (dev < 0 || dev >= 64 || !configured[dev]) {
    cudaError_t e = cudaFuncSetAttribute(attn_pair_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, PC::SMEM_BYTES);
    if (e != cudaSuccess) return e;
    if (dev >= 0 && dev < 64) configured[dev] = true;
  }
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)(2 * p.max_splits * p.max_row_groups), (unsigned)p.n_kv_heads, (unsigned)(p.n_layers * p.n_tasks));
  cfg.blockDim = dim3(PC::NTHREADS, 1, 1);
  cfg.dynamicSmemBytes = PC::SMEM_BYTES;
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, attn_pair_kernel, p, *tm_k, *tm_v);
}

}  // namespace fcg
