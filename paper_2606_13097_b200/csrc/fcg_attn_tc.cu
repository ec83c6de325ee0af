// S6: tensor-core patch attention on tcgen05 / TMEM (cache-patching, Eq. 6, PAPER.md:118-123, 718;
// DESIGN.md "Kernel S6").  Default attention path for both head dims (128: two 64-column operand halves per tile;
// 64: one): short patches and decode steps (HBM-bound) as well as long patches (tensor-bound).
//
//   CTA   = (KV split x row group of NQ*128 rows, kv head, layer x task), 1 CTA / SM, template <NQ, PS>:
//             <1,1>  one 128-row Q tile; R <= 64 rows are held 2x / 4x ("row streams": stream s owns the columns
//                    [s*NC, (s+1)*NC) of every KV tile with its own (m, l, O)), merged by log-sum-exp at the end
//             <1,2>  one Q tile, two softmax warpgroups on alternating KV tiles ("tile-parity streams")
//             <2,1>  two Q tiles, one softmax warpgroup each (K/V read once per 256 rows)
//   softmax warps    thread == query row == TMEM lane.  S tile read with tcgen05.ld, online softmax in the exp2
//                    domain with a lazy (threshold 2^8) O rescale, packed fp32 pairs;
//                    P goes back to TMEM as packed bf16 (tcgen05.st) -- with two Q tiles in place, over the
//                    first half of its S tile
//   K / V loader     one warp each: a TMA box copy (cp.async.bulk.tensor.5d, 128B swizzle) per (page, 64-column
//                    half) through the page table into a ring of 64-token tiles; transaction-count mbarriers
//   MMA warp         tcgen05.mma, M = 128, kind::f16, fp32 accumulate, issued from uniform registers:
//                    S[t][j&1] = Q_t K_j^T (N = 64, K = 128, operands in shared memory, K-major) and
//                    O += P_j V_j (N = 128, K = 64, A = P from TMEM, B = V MN-major from shared memory)
//   TMEM  (512 columns)  NQ = 1: S[b] at b*64, O[stream] at 128 + stream*128, P[b] at 384 + b*32
//                        NQ = 2: S[t][b] at (2t+b)*64 (P inside it), O_t at 256 + t*128
//   Tail  : tokens >= the end of the split inside the last tile are never valid data (page slack or
//           stale shared memory).  Their S columns are masked by selection; their V rows are zeroed
//           in shared memory by the MMA warp before P V, so no 0 x NaN can reach O.
//   Output: final bf16 rows (one split) or fp32 (m, l, o) partials for attn_combine_kernel.
#include <cuda_bf16.h>

#include <type_traits>

#include "fcg_internal.h"
#include "fcg_tc_common.cuh"

namespace fcg {
namespace {

constexpr int BM = 128;        // query rows per Q tile (UMMA M)
constexpr int BN = 64;         // cache tokens per K/V tile
constexpr float RESCALE_TAU = 8.0f;   // log2 units: keep a stale row max while the new one is < 2^8 larger

// ---- shared memory map -------------------------------------------------------------------------
// D = head_dim (64, 128 or 256): a tile is D / 64 halves of 64 columns, each [rows][128 B] with the 128B swizzle
template <int NQ, int PS_, int D_>
struct Cfg {
  static constexpr int D = D_;
  static constexpr int CPR = D / 8;                     // 16-byte chunks per row
  static constexpr int Q_TILE_B = BM * D * 2;
  static constexpr int KV_TILE_B = BN * D * 2;
  // separate rings: a K stage is free again as soon as Q K^T of its tile has completed, a V stage only after P V
  // P (the A operand of P V) lives in TMEM: the softmax threads write it with tcgen05.st and the MMA reads it from
  // there, so it never crosses shared memory (whose bandwidth -- Q, K, P, V operand reads plus the TMA and P writes,
  // 224 KB per 64-token step with two Q tiles -- was the limiter of the tensor-bound class).  One Q tile: own
  // columns; two Q tiles: P overwrites the first half of its S tile in place (S is then freed by P V, not by s_free).
  static constexpr bool P_ALIAS = NQ == 2;
  // head_dim 64, one Q tile, one softmax warpgroup (the short-patch / decode class): TWO CTAs per SM -- a 64-token tile
  // is only 16 KB there, so the per-tile latency chain (S ready -> softmax -> P ready -> P V) of a single CTA cannot
  // keep the SM's share of HBM busy; two independent CTAs hide each other's.  Each takes half the shared memory
  // (6 + 5 stages of 8 KB) and 256 TMEM columns (S 2 x 64, O 64, P 2 x 32).
  static constexpr int CTAS_PER_SM = (D == 64 && NQ == 1 && PS_ == 1) ? 2 : 1;
  // head_dim 256 (one Q tile only: O alone takes 256 TMEM columns): Q 64 KB + 3 K stages + 2 V stages of 32 KB
  static constexpr int K_STAGES = D == 256 ? 3 : (CTAS_PER_SM == 2 ? 6 : (NQ == 1 ? 6 : 5) * (128 / D));   // else the same bytes in flight for either head_dim
  static constexpr int V_STAGES = D == 256 ? 2 : (CTAS_PER_SM == 2 ? 5 : (NQ == 1 ? 6 : 5) * (128 / D));
  static_assert(D != 256 || (NQ == 1 && PS_ == 1), "head_dim 256: S 2 x 64 + O 256 + P 2 x 32 TMEM columns leave room for one Q tile and one stream set");
  // Tile-parity streams (NQ == 1 only): two softmax warpgroups, group w owns the KV tiles j = w (mod 2), its own
  // S / P buffer and its own O accumulator, with its own running (m, l); the streams are merged by log-sum-exp in
  // the epilogue like the row streams.  Two softmax warps per SM sub-partition hide each other's latencies.
  static constexpr int PS = PS_;
  static_assert(PS == 1 || (PS == 2 && NQ == 1), "parity streams need the TMEM columns of the second Q tile");
  static constexpr int N_SOFTMAX = 128 * NQ * PS;       // (Q tile | parity stream) x 4 lane quarters x 32 rows
  static constexpr int NTHREADS = N_SOFTMAX + 96;
  static constexpr int KLOAD_WARP = N_SOFTMAX / 32, VLOAD_WARP = KLOAD_WARP + 1, MMA_WARP = KLOAD_WARP + 2;
  static constexpr int TMEM_COLS = CTAS_PER_SM == 2 ? 256 : 512;   // S: 2*NQ x 64 columns, O: NQ*PS x 128 columns
  static constexpr int TMEM_O = NQ * 128;               // first O column
  static constexpr int Q_ITERS = NQ * BM * CPR / N_SOFTMAX;
  static constexpr int OFF_Q = 0;
  static constexpr int OFF_K = OFF_Q + NQ * Q_TILE_B;                // K stage s at +s*KV_TILE_B
  static constexpr int OFF_V = OFF_K + K_STAGES * KV_TILE_B;         // V stage s at +s*KV_TILE_B
  static constexpr int OFF_BAR = OFF_V + V_STAGES * KV_TILE_B;
  static constexpr int TMEM_P = CTAS_PER_SM == 2 ? 192 : 384;   // one Q tile: P[b] at TMEM_P + b*32 (S 0..127, O from 128)
  // k_full[SK], k_empty[SK], v_full[SV], v_empty[SV], s_full[NQ][2], p_full[NQ][2], pv_done[NQ][2], s_free[NQ][2],
  // q_full, all_done
  static constexpr int N_BARS = 2 * K_STAGES + 2 * V_STAGES + 8 * NQ + 2;
  static constexpr int SMEM_BYTES = OFF_BAR + N_BARS * 8 + 16 + 1024;   // + tmem slot + alignment slack
  static constexpr int MROW = D + 4;                    // fp32 row stride of the merge buffer: conflict-free 16-B accesses
  static_assert((K_STAGES + V_STAGES) * KV_TILE_B >= PS * BM * MROW * 4 + PS * BM * 8, "merge buffer must fit in the idle rings");
};

// The whole CTA program for one work item (task, layer index, kv head, KV split, row group).  Called by the per-class
// kernels below (indices from the 3-D grid) and by attn_tc_mixed_kernel (indices from an item table); a CTA may have
// more warps than this class uses (mixed kernel): those take no role and only meet the two CTA-wide barriers.
// PAD: the real head_dim d = p.head_dim is a multiple of 16 below the instantiated D (R27): Q rows and output rows have d
// elements, the Q tile's columns [d, D) are zero, and the K / V boxes come from a tensor map whose innermost extent is d, so
// TMA zero-fills their columns [d, D) -- the MMAs run at D, the zero columns add nothing to S and give zero O columns.
template <int NQ, int PS_, int D, bool PAD = false>
__device__ __forceinline__ void attn_tc_body(const AttnParams &p, const TmaDesc &tm_k, const TmaDesc &tm_v, unsigned char *smem_raw,
                                             const int task_i, const int li, const int g, const int split, const int rg) {
  using C = Cfg<NQ, PS_, D>;
  constexpr int SK = C::K_STAGES, SV = C::V_STAGES, PS = C::PS;
  constexpr int Q_TILE_B = C::Q_TILE_B, KV_TILE_B = C::KV_TILE_B, CPR = C::CPR;
  // 1024-byte alignment for the 128B-swizzle atoms
  unsigned char *smem = reinterpret_cast<unsigned char *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  const uint32_t sbase = smem_u32(smem);

  const AttnTaskDev tk = p.tasks[task_i];
  const int G = p.group;
  const int R = tk.n * G;
  const int row0 = rg * (NQ * BM);                 // first query row of this CTA
  if (split >= tk.n_splits || row0 >= R) return;
  const int layer = p.layer_begin + li;
  const int tid = threadIdx.x, lane = tid & 31;
  const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);   // tells the compiler that the warp index is warp-uniform
  const int d = PAD ? p.head_dim : D;                       // elements per q / out row
  // row -> (token, head in group) without a division per Q vector: r / G = umulhi(r, 2^32 / G + 1), exact while r * G < 2^32
  // (rows per kv head stay far below that).  The 16 address computations of a thread's Q loads, two runtime divisions each,
  // were 3.5 us of every CTA's prologue (globaltimer: softmax branch entered at 0.9 us, Q in registers at 4.4 us).
  const uint32_t g_magic = G > 1 ? (uint32_t)((1ull << 32) / (uint32_t)G + 1) : 0u;
  auto row_tok = [&](int r) -> int { return G > 1 ? (int)__umulhi((uint32_t)r, g_magic) : r; };

  // ---- row layout of this CTA (see "Row streams" in the header) ---------------------------------
  const int Rc = min(R - row0, NQ * BM);           // valid query rows of this CTA
  const int nq_eff = (NQ == 2 && Rc > BM) ? 2 : 1; // Q tiles that hold any valid row
  // row streams only with one Q tile per CTA: with two, P overwrites its S tile in TMEM, which leaves no zeroed columns
  // for the slices a stream does not own (a trailing row group of <= 64 rows simply runs with idle lanes)
  const int dup = NQ == 1 ? (Rc <= 32 ? 4 : (Rc <= 64 ? 2 : 1)) : 1;
  const int rps = BM / dup;                        // MMA rows per stream (128, 64 or 32)

  const int t_begin = split * tk.split_len;
  const int t_end = min(tk.kv_len, t_begin + tk.split_len);
  const int32_t *pos = p.positions + tk.tok_off;
  const int cta_last = row0 + Rc - 1;
  const int cta_max_lim = min(pos[cta_last / G], t_end - 1);
  const int n_tiles = cta_max_lim >= t_begin ? (cta_max_lim - t_begin) / BN + 1 : 0;

  const uint32_t bar0 = sbase + C::OFF_BAR;
  auto k_full = [&](int s) { return bar0 + 8 * s; };
  auto k_empty = [&](int s) { return bar0 + 8 * (SK + s); };
  auto v_full = [&](int s) { return bar0 + 8 * (2 * SK + s); };
  auto v_empty = [&](int s) { return bar0 + 8 * (2 * SK + SV + s); };
  constexpr int B0 = 2 * SK + 2 * SV;
  auto s_full = [&](int t, int b) { return bar0 + 8 * (B0 + 2 * t + b); };
  auto p_full = [&](int t, int b) { return bar0 + 8 * (B0 + 2 * NQ + 2 * t + b); };
  auto pv_done = [&](int t, int b) { return bar0 + 8 * (B0 + 4 * NQ + 2 * t + b); };
  auto s_free = [&](int t, int b) { return bar0 + 8 * (B0 + 6 * NQ + 2 * t + b); };
  const uint32_t q_full = bar0 + 8 * (B0 + 8 * NQ);
  const uint32_t all_done = bar0 + 8 * (B0 + 8 * NQ + 1);
  const uint32_t tmem_slot = bar0 + 8 * C::N_BARS;
  volatile uint32_t *tmem_slot_ptr = reinterpret_cast<volatile uint32_t *>(smem + C::OFF_BAR + 8 * C::N_BARS);

  // valid rows of Q tile t, and its softmax warps that own at least one valid row (the others never
  // touch the tile's barriers: the P-ready barrier counts the threads of the active warps only)
  auto tile_rows = [&](int t) { return max(0, min(Rc - t * BM, BM)); };
  auto warp_active = [&](int t, int w) { return ((32 * w) & (rps - 1)) < tile_rows(t); };

  if (tid == 0) {
    for (int s = 0; s < SK; ++s) {
      mbar_init(k_full(s), 1);
      mbar_init(k_empty(s), 1);
    }
    for (int s = 0; s < SV; ++s) {
      mbar_init(v_full(s), 1);
      mbar_init(v_empty(s), 1);
    }
    for (int t = 0; t < NQ; ++t) {
      int act = 0;
      for (int w = 0; w < 4; ++w) act += warp_active(t, w) ? 1 : 0;
      for (int b = 0; b < 2; ++b) {
        mbar_init(s_full(t, b), 1);
        mbar_init(p_full(t, b), 32 * max(act, 1));
        mbar_init(s_free(t, b), 32 * max(act, 1));
        mbar_init(pv_done(t, b), 1);
      }
    }
    mbar_init(q_full, C::N_SOFTMAX);
    mbar_init(all_done, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == C::MMA_WARP) tmem_alloc<C::TMEM_COLS>(tmem_slot);
  if (warp == C::KLOAD_WARP && lane == 0) tma_prefetch_desc(&tm_k);
  if (warp == C::VLOAD_WARP && lane == 0) tma_prefetch_desc(&tm_v);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  // shuffle broadcast: the value is warp-uniform, and saying so keeps every TMEM address of the MMA warp in uniform
  // registers (the MMA warp was issue-bound: ~255 SASS instructions per KV tile, a third of them R2UR / UMOV)
  const uint32_t tmem_base = __shfl_sync(0xffffffffu, *tmem_slot_ptr, 0);
  // programmatic dependent launch: everything above (barrier init, TMEM allocation, tensor-map prefetch) may overlap the
  // scatter kernel that precedes this launch; the cache rows it writes are only read below.  A no-op when the
  // launch does not carry the attribute.  The combine kernel that may follow is allowed to pre-launch right away.
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");

  if (warp == C::KLOAD_WARP || warp == C::VLOAD_WARP) {
    // ======================================= loaders =======================================
    // One warp streams K, one streams V: lanes 0..ppt-1 look up the pages of the NEXT tile (coalesced, latency
    // hidden behind the ring wait); one elected lane then issues two box copies per page (the two 64-column
    // halves).  K and V are separate instantiations so that everything but the page id is warp-uniform at compile
    // time (tensor map, ring and barrier addresses stay in uniform registers; UTMALDG takes uniform operands).
    auto load_stream = [&](auto is_k_tag) {
      constexpr bool is_k = decltype(is_k_tag)::value;
      const TmaDesc *tm = is_k ? &tm_k : &tm_v;
      constexpr int NS = is_k ? SK : SV;
      const uint32_t ring = sbase + (is_k ? C::OFF_K : C::OFF_V);
      const uint32_t full0 = is_k ? k_full(0) : v_full(0), empty0 = is_k ? k_empty(0) : v_empty(0);
      const int P = p.page_size;
      const int pshift = __ffs(P) - 1;
      const int ppt = BN >> pshift;                   // pages per tile (P <= 64, power of two)
      const int32_t *table = p.tables + tk.table_off + (t_begin >> pshift);
      const int n_pages_split = (t_end - t_begin + P - 1) >> pshift;
      auto page_of = [&](int j) -> int {
        const int pi = j * ppt + lane;
        return (lane < ppt && pi < n_pages_split) ? __ldg(table + pi) : -1;
      };
      int page = page_of(0);
      int st = 0, round = 0;
      for (int j = 0; j < n_tiles; ++j) {
        const int page_next = page_of(j + 1);
        if (round > 0) mbar_wait(empty0 + 8 * st, (round - 1) & 1);
        const int n_ok = min(ppt, n_pages_split - j * ppt);
        const uint32_t dst = ring + st * KV_TILE_B;
        const uint32_t bar = full0 + 8 * st;
        if (elect_one()) mbar_arrive_expect_tx(bar, (uint32_t)(n_ok * P * (D * 2)));
#pragma unroll 1
        for (int i = 0; i < n_ok; ++i) {
          const int pg = __shfl_sync(0xffffffffu, page, i);
#pragma unroll
          for (int h = 0; h < D / 64; ++h) tma_load_5d(dst + i * P * 128 + h * (BN * 128), tm, bar, 64 * h, 0, g, pg, layer);
        }
        page = page_next;
        if (++st == NS) {
          st = 0;
          ++round;
        }
      }
    };
    if (warp == C::KLOAD_WARP)
      load_stream(std::true_type{});
    else
      load_stream(std::false_type{});
  } else if (warp == C::MMA_WARP) {
    // ======================================= MMA issuer =====================================
    if (n_tiles > 0) {
      constexpr uint32_t IDESC_S = idesc_f16(BN, false);
      constexpr uint32_t IDESC_O = idesc_f16(D, true);
      mbar_wait(q_full, 0);
      // operand descriptors: a fixed part per operand, plus (byte offset >> 4) in the 14-bit address field
      const uint64_t qdesc0 = smem_desc(sbase + C::OFF_Q, 16, 1024);
      const uint64_t kdesc0 = smem_desc(sbase + C::OFF_K, 16, 1024);
      const uint64_t vdesc0 = smem_desc(sbase + C::OFF_V, BN * 128, 1024);   // MN-major: LBO = next 64-column half
      int sk = 0, rk = 0;                            // K ring position of the next Q K^T
      auto issue_qk = [&](int j) {
        // S[t][j&1] was last read by the softmax of tile j-2: reuse it as soon as those threads have loaded it -- or,
        // where P sits inside the S tile, once P V of tile j-2 has consumed it
        if (!C::P_ALIAS && j >= 2) {
#pragma unroll
          for (int t = 0; t < NQ; ++t)
            if (t < nq_eff) mbar_wait(s_free(t, j & 1), ((j - 2) >> 1) & 1);
        }
        mbar_wait(k_full(sk), rk & 1);
        const uint64_t kdesc = kdesc0 + (uint64_t)((sk * KV_TILE_B) >> 4);
        tc_fence_after();
#pragma unroll
        for (int t = 0; t < NQ; ++t) {
          if (t < nq_eff) {
            // P inside S: wait for P V of tile j-2 of THIS Q tile only, right before overwriting its S -- the other Q
            // tile's MMAs keep the tensor pipe busy meanwhile (no drain between P V and Q K^T)
            if (C::P_ALIAS && j >= 2) {
              mbar_wait(pv_done(t, j & 1), ((j - 2) >> 1) & 1);
              tc_fence_after();
            }
#pragma unroll
            for (int k = 0; k < D / 16; ++k) {
              const uint64_t a = qdesc0 + (uint64_t)((t * Q_TILE_B + (k >> 2) * (BM * 128) + (k & 3) * 32) >> 4);
              const uint64_t b = kdesc + (uint64_t)(((k >> 2) * (BN * 128) + (k & 3) * 32) >> 4);
              umma_ss(tmem_base + (2 * t + (j & 1)) * BN, a, b, IDESC_S, k > 0);
            }
            umma_commit(s_full(t, j & 1));
          }
        }
        umma_commit(k_empty(sk));                    // the K stage is free once these MMAs have read it
        if (++sk == SK) {
          sk = 0;
          ++rk;
        }
      };
      int sv = 0, rv = 0;
      auto issue_pv = [&](int j) {
        mbar_wait(v_full(sv), rv & 1);
        const int ts = t_begin + j * BN;
        if (ts + BN > t_end) {
          // ragged last tile: zero the V rows that hold no token of this split (whole warp)
          const int r0 = t_end - ts;
          unsigned char *vt = smem + C::OFF_V + sv * KV_TILE_B;
          for (int i = lane; i < (BN - r0) * CPR; i += 32) {
            const int row = r0 + i / CPR, c = i % CPR;
            *reinterpret_cast<uint4 *>(vt + (c >> 3) * (BN * 128) + row * 128 + ((c & 7) << 4)) = make_uint4(0, 0, 0, 0);
          }
          fence_proxy_async();
          __syncwarp();
        }
        const uint64_t vdesc = vdesc0 + (uint64_t)((sv * KV_TILE_B) >> 4);
#pragma unroll
        for (int t = 0; t < NQ; ++t) {
          if (t < nq_eff) {
            mbar_wait(p_full(t, j & 1), (j >> 1) & 1);
            tc_fence_after();
            const uint32_t tmem_p = tmem_base + (C::P_ALIAS ? (2 * t + (j & 1)) * BN : C::TMEM_P + (j & 1) * 32);
            // O accumulator of (Q tile t | parity stream j % PS); the stream's first tile overwrites it
            const uint32_t tmem_o = tmem_base + C::TMEM_O + (PS == 2 ? (j & 1) : t) * 128;
#pragma unroll
            for (int k = 0; k < BN / 16; ++k)
              umma_ts(tmem_o, tmem_p + k * 8, vdesc + (uint64_t)((k * 2048) >> 4), IDESC_O, (j >= PS || k > 0) ? 1u : 0u);
            if (t == nq_eff - 1) umma_commit(v_empty(sv));
            umma_commit(pv_done(t, j & 1));
          }
        }
        if (++sv == SV) {
          sv = 0;
          ++rv;
        }
      };
      // Issue order = expected order of the events waited for.  One stream: S(j) loaded, P(j) written, S(j+1)
      // loaded, ...  Two parity streams run half a tile apart: S(j) loaded, P(j-1) written, S(j+1) loaded, ...
      constexpr int LAG = PS - 1;
      issue_qk(0);
      if (n_tiles > 1) issue_qk(1);
      for (int j = 0; j < n_tiles; ++j) {
        if (C::P_ALIAS) {
          // P sits inside S[j&1]: Q K^T of tile j+2 may only overwrite it after P V of tile j
          issue_pv(j);
          if (j + 2 < n_tiles) issue_qk(j + 2);
        } else {
          if (j + 2 < n_tiles) issue_qk(j + 2);
          if (j >= LAG) issue_pv(j - LAG);
        }
      }
      for (int j = max(0, n_tiles - LAG); j < n_tiles; ++j) issue_pv(j);
      umma_commit(all_done);
    }
  } else if (warp < C::N_SOFTMAX / 32) {
    // ======================================= softmax ========================================
    // Q tiles: MMA row m of tile t holds query row  row0 + t*BM + (m % rps)  -> (token, head-in-group); with
    // dup > 1 the same query rows are replicated `dup` times (one copy per stream); rows past the valid ones
    // are zero.  All softmax threads copy cooperatively (coalesced 16-B chunks), then hand Q to the MMA thread.
    // All 16 loads of a thread are issued before the first store: one global-memory round trip per CTA
    // instead of sixteen (the round-1 capture had 16 % of a softmax warp's life in this prologue).
    constexpr int Q_BATCH = C::Q_ITERS > 16 ? 16 : C::Q_ITERS;    // head_dim 256: two batches of 16 loads (64 registers each)
#pragma unroll
    for (int i0 = 0; i0 < C::Q_ITERS; i0 += Q_BATCH) {
      uint4 qv[Q_BATCH];
#pragma unroll
      for (int i = 0; i < Q_BATCH; ++i) {
        const int ci = tid + C::N_SOFTMAX * (i0 + i);
        const int row = ci / CPR, c = ci % CPR;
        const int rt = row & (BM - 1), tq = row >> 7;
        const int rl = rt & (rps - 1);
        qv[i] = make_uint4(0, 0, 0, 0);
        if (rl < tile_rows(tq) && (!PAD || c * 8 < d)) {
          const int r = row0 + tq * BM + rl;
          const int rtok = row_tok(r);
          const uint16_t *src = p.q + (((size_t)li * p.n_total + tk.tok_off + rtok) * p.n_q_heads + g * G + (r - rtok * G)) * d + c * 8;
          qv[i] = __ldg(reinterpret_cast<const uint4 *>(src));
        }
      }
#pragma unroll
      for (int i = 0; i < Q_BATCH; ++i) {
        const int ci = tid + C::N_SOFTMAX * (i0 + i);
        const int row = ci / CPR, c = ci % CPR;
        const int rt = row & (BM - 1), tq = row >> 7;
        const uint32_t dst = C::OFF_Q + tq * Q_TILE_B + (c >> 3) * (BM * 128) + rt * 128 + (((c & 7) ^ (rt & 7)) << 4);
        *reinterpret_cast<uint4 *>(smem + dst) = qv[i];
      }
    }
    const int wg = warp >> 2;                  // softmax warpgroup: the Q tile (NQ == 2) or the parity stream (NQ == 1)
    const int qt = PS == 2 ? 0 : wg;           // Q tile of this warp
    const int par = PS == 2 ? wg : 0;          // parity stream of this warp: KV tiles j = par (mod PS)
    const int row = tid & (BM - 1);            // MMA row in the tile == TMEM lane
    const uint32_t lane_addr = ((uint32_t)((warp & 3) * 32) << 16);
    if (!C::P_ALIAS && dup > 1) {
      // a stream writes only its own columns of P: the rest of the row stays zero for the whole kernel
      uint32_t zero[32];
#pragma unroll
      for (int c = 0; c < 32; ++c) zero[c] = 0u;
      TMEM_ST_32(tmem_base + lane_addr + C::TMEM_P + par * 32, zero);
      if (PS == 1) TMEM_ST_32(tmem_base + lane_addr + C::TMEM_P + 32, zero);
      tmem_wait_st();
      tc_fence_before();
    }
    fence_proxy_async();
    mbar_arrive(q_full);

    const int strm = row / rps;                // row stream of this thread: columns [strm*NC, strm*NC + NC) of every tile
    const int rl = row & (rps - 1);
    const int r = row0 + qt * BM + rl;
    const bool tile_used = qt < nq_eff;
    const bool active = tile_used && warp_active(qt, warp & 3);
    const bool valid = tile_used && rl < tile_rows(qt);
    const int lim = valid ? min(pos[r / G], t_end - 1) : -1;
    const uint32_t tmem_s = tmem_base + lane_addr + (2 * qt) * BN;
    const uint32_t tmem_o = tmem_base + lane_addr + C::TMEM_O + wg * 128;
    const float sc = p.scale_log2;
    float m_ref = -INFINITY;                   // reference max used for exp2 (may lag the true max by < TAU)
    float l = 0.f;

    auto softmax_tiles = [&](auto nc_tag) {
      constexpr int NC = decltype(nc_tag)::value;       // S columns per thread and tile
      const int c0 = strm * NC;
      for (int j = par; j < n_tiles; j += PS) {
        const int ts = t_begin + j * BN + c0;           // token of this thread's first column
        const int b = j & 1;
        mbar_wait(s_full(qt, b), (j >> 1) & 1);
        tc_fence_after();
        uint32_t sreg[NC];
        if constexpr (NC == 64) {
          TMEM_LD_32(tmem_s + b * BN, sreg);
          TMEM_LD_32(tmem_s + b * BN + 32, (sreg + 32));
        } else if constexpr (NC == 32) {
          TMEM_LD_32(tmem_s + b * BN + c0, sreg);
        } else {
          TMEM_LD_16(tmem_s + b * BN + c0, sreg);
        }
        tmem_wait_ld();
        if (!C::P_ALIAS) {
          tc_fence_before();
          mbar_arrive(s_free(qt, b));                   // S[b] may be overwritten by Q K^T of tile j+2
        }
        if (ts + NC - 1 > lim) {
#pragma unroll
          for (int c = 0; c < NC; ++c)
            if (ts + c > lim) sreg[c] = 0xff800000u;     // -inf, by selection (S may be garbage there)
        }
        float mx4[4] = {-INFINITY, -INFINITY, -INFINITY, -INFINITY};
#pragma unroll
        for (int c = 0; c < NC; ++c) mx4[c & 3] = fmaxf(mx4[c & 3], __uint_as_float(sreg[c]));
        const float mx = fmaxf(fmaxf(mx4[0], mx4[1]), fmaxf(mx4[2], mx4[3]));
        const float m_new = fmaxf(m_ref, mx * sc);
        // lazy rescale: move the reference only when it is too far behind
        float factor = 1.f;
        const bool bump = (m_new - m_ref > RESCALE_TAU) || (m_ref == -INFINITY && m_new != -INFINITY);
        if (bump) {
          factor = (m_ref == -INFINITY) ? 0.f : ex2_approx(m_ref - m_new);
          m_ref = m_new;
        }
        if (j >= PS && __any_sync(0xffffffffu, bump)) {
          // O holds the stream's earlier tiles only once P V of its previous tile j-PS has completed
          mbar_wait(pv_done(qt, (j - PS) & 1), ((j - PS) >> 1) & 1);
          tc_fence_after();
#pragma unroll
          for (int ch = 0; ch < D / 32; ++ch) {
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
        // the P buffer of this parity was last read by P V of tile j-2 (implied when P sits inside S: Q K^T of this
        // tile was only issued after that P V)
        if (!C::P_ALIAS && j >= 2) mbar_wait(pv_done(qt, b), ((j - 2) >> 1) & 1);
        uint32_t preg[NC / 2];
        // packed fp32 pairs (FFMA2 / FADD2) for the scale-subtract and the row sum; every exp2 on the MUFU (moving a
        // share of them to a polynomial on the FMA pipe cost more issue slots than the MUFU time it saved)
        const float2 sc2 = make_float2(sc, sc), nmu2 = make_float2(-mu, -mu);
        float2 sum2[2] = {make_float2(0.f, 0.f), make_float2(0.f, 0.f)};
#pragma unroll
        for (int c8 = 0; c8 < NC / 8; ++c8) {
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
        // P row -> TMEM (row == lane, two bf16 per column): this stream's slice of the 32 packed columns
        const uint32_t tmem_p = tmem_base + lane_addr + (C::P_ALIAS ? (2 * qt + b) * BN : C::TMEM_P + b * 32) + (c0 >> 1);
        if constexpr (NC == 64) {
          TMEM_ST_32(tmem_p, preg);
        } else if constexpr (NC == 32) {
          TMEM_ST_16(tmem_p, preg);
        } else {
          TMEM_ST_8(tmem_p, preg);
        }
        tmem_wait_st();
        tc_fence_before();
        mbar_arrive(p_full(qt, b));
      }
    };
    if (active) {
      if (dup == 1)
        softmax_tiles(std::integral_constant<int, 64>{});
      else if (dup == 2)
        softmax_tiles(std::integral_constant<int, 32>{});
      else
        softmax_tiles(std::integral_constant<int, 16>{});
    }

    // ---- epilogue: merge the streams, then O / l -> bf16, or partials ---------------------------
    // all_done completes when every MMA of the CTA has: the accumulators are final and the K/V rings (which the
    // merge buffer reuses) are idle.  A stream without any tile (n_tiles <= par) contributes (m, l) = (-inf, 0).
    const bool have_o = active && n_tiles > par;
    if (n_tiles > 0) {
      mbar_wait(all_done, 0);
      tc_fence_after();
    }
    constexpr int MROW = C::MROW;
    float *mbuf = reinterpret_cast<float *>(smem + C::OFF_K);                              // [PS*BM][MROW], over the idle K/V rings
    float2 *mlbuf = reinterpret_cast<float2 *>(smem + C::OFF_K + PS * BM * MROW * 4);     // [PS*BM] (m, l)
    const int n_streams = dup * PS;                // streams holding a copy of each query row (Q tile 0 only)
    const bool merging = n_streams > 1 && qt == 0;
    const bool lead = strm == 0 && par == 0;       // the stream that merges and writes the row
    const int mrow = par * BM + row;               // this thread's row in the merge buffer
    if (merging) {
      if (!lead && active) {
#pragma unroll
        for (int ch = 0; ch < D / 32; ++ch) {
          uint32_t oreg[32];
          if (have_o) {
            TMEM_LD_32(tmem_o + ch * 32, oreg);
            tmem_wait_ld();
          } else {
#pragma unroll
            for (int c = 0; c < 32; ++c) oreg[c] = 0u;
          }
#pragma unroll
          for (int c = 0; c < 32; c += 4)
            *reinterpret_cast<uint4 *>(mbuf + mrow * MROW + ch * 32 + c) = make_uint4(oreg[c], oreg[c + 1], oreg[c + 2], oreg[c + 3]);
        }
        mlbuf[mrow] = make_float2(m_ref, l);
      }
      // the softmax warps that share Q tile 0: all eight with parity streams, else the tile's four
      if (PS == 2)
        asm volatile("bar.sync 1, 256;" ::: "memory");
      else
        asm volatile("bar.sync 1, 128;" ::: "memory");   // NQ == 2: only the four warps of Q tile 0 get here
    }
    float w_own = 1.f, w_oth[8];
    float m_out = m_ref, l_out = l;
    const bool writer = valid && lead;
    if (writer && merging) {
      // streams other than the lead: (parity sp, row stream ss) -> merge-buffer row sp*BM + ss*rps + rl
      float M = m_ref;
      for (int s = 1; s < n_streams; ++s) M = fmaxf(M, mlbuf[(s / dup) * BM + (s % dup) * rps + rl].x);
      const float Mu = M == -INFINITY ? 0.f : M;
      w_own = ex2_approx(m_ref - Mu);              // exp2(-inf) = 0 for a stream that saw nothing
      float L = w_own * l;
      for (int s = 1; s < n_streams; ++s) {
        const float2 ml = mlbuf[(s / dup) * BM + (s % dup) * rps + rl];
        w_oth[s] = ex2_approx(ml.x - Mu);
        L += w_oth[s] * ml.y;
      }
      m_out = M;
      l_out = L;
    }
    const int i_tok = writer ? r / G : 0, hh = writer ? r % G : 0;
    const size_t out_row = ((size_t)li * p.n_total + tk.tok_off + i_tok) * p.n_q_heads + g * G + hh;
    const size_t prow_i = ((size_t)(li * p.max_splits + split) * p.n_total + tk.tok_off + i_tok) * p.n_q_heads + g * G + hh;
    const bool final_out = tk.n_splits == 1;
    const float inv = l_out > 0.f ? 1.f / l_out : 0.f;
    if (lead && active) {
#pragma unroll
      for (int ch = 0; ch < D / 32; ++ch) {
        uint32_t oreg[32];
        if (have_o) {
          TMEM_LD_32(tmem_o + ch * 32, oreg);
          tmem_wait_ld();
        } else {
#pragma unroll
          for (int c = 0; c < 32; ++c) oreg[c] = 0u;
        }
        if (writer) {
          float o[32];
#pragma unroll
          for (int c = 0; c < 32; ++c) o[c] = __uint_as_float(oreg[c]);
          if (merging) {
#pragma unroll
            for (int c = 0; c < 32; ++c) o[c] *= w_own;
            for (int s = 1; s < n_streams; ++s) {
              const float *src = mbuf + ((s / dup) * BM + (s % dup) * rps + rl) * MROW + ch * 32;
              const float w = w_oth[s];
#pragma unroll
              for (int c = 0; c < 32; c += 4) {
                const float4 x = *reinterpret_cast<const float4 *>(src + c);
                o[c] = fmaf(w, x.x, o[c]);
                o[c + 1] = fmaf(w, x.y, o[c + 1]);
                o[c + 2] = fmaf(w, x.z, o[c + 2]);
                o[c + 3] = fmaf(w, x.w, o[c + 3]);
              }
            }
          }
          if (final_out) {
            uint16_t *dst = p.out + out_row * d + ch * 32;
#pragma unroll
            for (int c = 0; c < 32; c += 8) {
              if (PAD && ch * 32 + c >= d) break;
              uint4 v;
              v.x = pack_bf16(o[c] * inv, o[c + 1] * inv);
              v.y = pack_bf16(o[c + 2] * inv, o[c + 3] * inv);
              v.z = pack_bf16(o[c + 4] * inv, o[c + 5] * inv);
              v.w = pack_bf16(o[c + 6] * inv, o[c + 7] * inv);
              *reinterpret_cast<uint4 *>(dst + c) = v;
            }
          } else {
            float *dst = p.part_o + prow_i * d + ch * 32;
#pragma unroll
            for (int c = 0; c < 32; c += 4) {
              if (PAD && ch * 32 + c >= d) break;
              *reinterpret_cast<float4 *>(dst + c) = make_float4(o[c], o[c + 1], o[c + 2], o[c + 3]);
            }
          }
        }
      }
      if (writer && !final_out) *reinterpret_cast<float2 *>(p.part_ml + prow_i * 2) = make_float2(m_out, l_out);
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == C::MMA_WARP) {
    tc_fence_after();
    tmem_dealloc<C::TMEM_COLS>(tmem_base);
  }
}

template <int NQ, int PS_, int D, bool PAD = false>
__global__ void __launch_bounds__(Cfg<NQ, PS_, D>::NTHREADS, Cfg<NQ, PS_, D>::CTAS_PER_SM)
    attn_tc_kernel(const AttnParams p, const __grid_constant__ TmaDesc tm_k, const __grid_constant__ TmaDesc tm_v) {
  extern __shared__ unsigned char smem_raw[];
  attn_tc_body<NQ, PS_, D, PAD>(p, tm_k, tm_v, smem_raw, blockIdx.z % p.n_tasks, blockIdx.z / p.n_tasks, blockIdx.y, blockIdx.x % p.max_splits,
                           blockIdx.x / p.max_splits);
}

// A batch that mixes the three CTA classes (C4: 8..64-token patches with G = 4 give 32..256 rows per kv head) in ONE
// launch: block b = hl * n_items + k runs item k (class, task, row group, split; p.items, interleaved proportionally
// over the classes by the host, longest task first inside a class) for (layer, kv head) hl.  One launch per class ran
// the classes back to back -- the HBM-bound ones (<= 128 rows) at the memory roofline with the tensor pipe half idle,
// then the compute-bound one (two Q tiles) with HBM half idle, each with its own tail; interleaved, CTAs of both kinds
// are resident at any time and share the machine.  head_dim 128 only (the head_dim-64 short-patch class lives on two
// CTAs per SM, which a kernel sized for the largest class cannot offer).
constexpr int MIXED_THREADS = Cfg<2, 1, 128>::NTHREADS;
static_assert(Cfg<1, 2, 128>::NTHREADS == MIXED_THREADS && Cfg<1, 1, 128>::NTHREADS <= MIXED_THREADS, "the mixed kernel is sized for the largest class");
constexpr int MIXED_SMEM = Cfg<2, 1, 128>::SMEM_BYTES > Cfg<1, 2, 128>::SMEM_BYTES
                               ? (Cfg<2, 1, 128>::SMEM_BYTES > Cfg<1, 1, 128>::SMEM_BYTES ? Cfg<2, 1, 128>::SMEM_BYTES : Cfg<1, 1, 128>::SMEM_BYTES)
                               : (Cfg<1, 2, 128>::SMEM_BYTES > Cfg<1, 1, 128>::SMEM_BYTES ? Cfg<1, 2, 128>::SMEM_BYTES : Cfg<1, 1, 128>::SMEM_BYTES);

__global__ void __launch_bounds__(MIXED_THREADS, 1)
    attn_tc_mixed_kernel(const AttnParams p, const __grid_constant__ TmaDesc tm_k, const __grid_constant__ TmaDesc tm_v) {
  extern __shared__ unsigned char smem_raw[];
  const int hl = blockIdx.x / p.n_items;
  const int4 it = __ldg(p.items + (blockIdx.x - hl * p.n_items));      // {class, task index, row group, split}
  const int g = hl % p.n_kv_heads, li = hl / p.n_kv_heads;
  if (it.x == 2)
    attn_tc_body<2, 1, 128>(p, tm_k, tm_v, smem_raw, it.y, li, g, it.w, it.z);
  else if (it.x == 1)
    attn_tc_body<1, 2, 128>(p, tm_k, tm_v, smem_raw, it.y, li, g, it.w, it.z);
  else
    attn_tc_body<1, 1, 128>(p, tm_k, tm_v, smem_raw, it.y, li, g, it.w, it.z);
}

template <int NQ, int PS_, int D, bool PAD = false>
cudaError_t launch_nq(const AttnParams &p, const TmaDesc &tk, const TmaDesc &tv, cudaStream_t stream) {
  using C = Cfg<NQ, PS_, D>;
  // the attribute is per device (fcg_config_t.device allows libraries on several GPUs in one process)
  static bool configured[64] = {};
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess) return cudaGetLastError();
  if (dev < 0 || dev >= 64 || !configured[dev]) {
    cudaError_t e = cudaFuncSetAttribute(attn_tc_kernel<NQ, PS_, D, PAD>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_BYTES);
    if (e != cudaSuccess) return e;
    if (dev >= 0 && dev < 64) configured[dev] = true;
  }
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)(p.max_splits * p.max_row_groups), (unsigned)p.n_kv_heads, (unsigned)(p.n_layers * p.n_tasks));
  cfg.blockDim = dim3(C::NTHREADS, 1, 1);
  cfg.dynamicSmemBytes = C::SMEM_BYTES;
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, attn_tc_kernel<NQ, PS_, D, PAD>, p, tk, tv);
}

}  // namespace

// all CTA classes of a batch in one launch (head_dim 128): p.items / p.n_items list the work items, p.tasks all tasks
cudaError_t launch_attn_tc_mixed(const AttnParams &p, const TmaDesc *tm_k, const TmaDesc *tm_v, cudaStream_t stream) {
  if (!tm_k || !tm_v || !p.items || p.n_items <= 0) return cudaErrorInvalidValue;
  static bool configured[64] = {};
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess) return cudaGetLastError();
  if (dev < 0 || dev >= 64 || !configured[dev]) {
    cudaError_t e = cudaFuncSetAttribute(attn_tc_mixed_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, MIXED_SMEM);
    if (e != cudaSuccess) return e;
    if (dev >= 0 && dev < 64) configured[dev] = true;
  }
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)((size_t)p.n_items * p.n_kv_heads * p.n_layers), 1, 1);
  cfg.blockDim = dim3(MIXED_THREADS, 1, 1);
  cfg.dynamicSmemBytes = MIXED_SMEM;
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, attn_tc_mixed_kernel, p, *tm_k, *tm_v);
}

int attn_tc_ctas_per_sm(int head_dim, int q_tiles, int parity_streams) {
  return (head_dim <= 64 && q_tiles == 1 && parity_streams == 1) ? 2 : 1;
}

// q_tiles = 128-row Q tiles per CTA (1 or 2); p.max_row_groups counts groups of q_tiles*128 rows.
// parity_streams (q_tiles == 1 only): 2 = two softmax warpgroups on alternating KV tiles, 1 = one warpgroup.
cudaError_t launch_attn_tc(const AttnParams &p, int head_dim, int q_tiles, int parity_streams, const TmaDesc *tm_k,
                           const TmaDesc *tm_v, cudaStream_t stream) {
  if (head_dim < 16 || head_dim > 256 || head_dim % 16 || !tm_k || !tm_v || p.head_dim != head_dim) return cudaErrorNotSupported;
  if (head_dim == 256) {
    // one CTA class: a 128-row Q tile per CTA, more rows per kv head run as more row groups
    if (q_tiles == 1 && parity_streams == 1) return launch_nq<1, 1, 256>(p, *tm_k, *tm_v, stream);
  } else if (head_dim == 128) {
    if (q_tiles == 1 && parity_streams == 2) return launch_nq<1, 2, 128>(p, *tm_k, *tm_v, stream);
    if (q_tiles == 1) return launch_nq<1, 1, 128>(p, *tm_k, *tm_v, stream);
    if (q_tiles == 2) return launch_nq<2, 1, 128>(p, *tm_k, *tm_v, stream);
  } else if (head_dim == 64) {
    if (q_tiles == 1 && parity_streams == 2) return launch_nq<1, 2, 64>(p, *tm_k, *tm_v, stream);
    if (q_tiles == 1) return launch_nq<1, 1, 64>(p, *tm_k, *tm_v, stream);
    if (q_tiles == 2) return launch_nq<2, 1, 64>(p, *tm_k, *tm_v, stream);
  } else if (head_dim > 128) {
    // other multiples of 16 run the next instantiated width with zero-padded columns (PAD)
    if (q_tiles == 1 && parity_streams == 1) return launch_nq<1, 1, 256, true>(p, *tm_k, *tm_v, stream);
  } else if (head_dim > 64) {
    if (q_tiles == 1 && parity_streams == 2) return launch_nq<1, 2, 128, true>(p, *tm_k, *tm_v, stream);
    if (q_tiles == 1) return launch_nq<1, 1, 128, true>(p, *tm_k, *tm_v, stream);
    if (q_tiles == 2) return launch_nq<2, 1, 128, true>(p, *tm_k, *tm_v, stream);
  } else {
    if (q_tiles == 1 && parity_streams == 2) return launch_nq<1, 2, 64, true>(p, *tm_k, *tm_v, stream);
    if (q_tiles == 1) return launch_nq<1, 1, 64, true>(p, *tm_k, *tm_v, stream);
    if (q_tiles == 2) return launch_nq<2, 1, 64, true>(p, *tm_k, *tm_v, stream);
  }
  return cudaErrorInvalidValue;
}

}  // namespace fcg
