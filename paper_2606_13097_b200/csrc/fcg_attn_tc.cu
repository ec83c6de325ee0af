// S6: tensor-core patch attention on tcgen05 / TMEM (cache-patching, Eq. 6, PAPER.md:118-123, 718;
// DESIGN.md "Kernel S6").  Same result as the split-KV warp-MMA kernel, for R = n*G >= 64 query rows
// per kv head, where the two contractions Q K^T and P V are dense enough for the 5th-gen tensor cores.
//
//   CTA   = (KV split x row group of NQ*128 rows, kv head, layer x task); NQ*128 + 64 threads, 1 CTA / SM
//   warps [0, 4*NQ)  softmax: thread == query row == TMEM lane of its 128-row Q tile.  S tile read with
//                    tcgen05.ld, online softmax in the exp2 domain with a lazy (threshold 2^8) O rescale,
//                    P written as bf16 into a 128B-swizzled K-major shared tile (the A operand of P V)
//   warp  4*NQ       loader: one TMA box copy (cp.async.bulk.tensor.5d, 128B swizzle) per (page, K|V,
//                    64-column half) through the page table into a ring of 64-token K/V tiles; the
//                    transaction-count mbarrier of the stage completes when the bytes have landed, so
//                    loading is decoupled from the MMA / softmax chain
//   warp  4*NQ+1     MMA issuer: one thread issues tcgen05.mma (M=128, kind::f16, fp32 accumulate):
//                    S[t][j&1] = Q_t K_j^T (N=64, K=128, both K-major) and O_t += P_t,j V_j (N=128, K=64,
//                    V as an MN-major B operand), accumulators in TMEM.  Q K^T of tile j+1 is issued
//                    before P V of tile j, so the softmax of tile j overlaps tensor work.
//   TMEM  = S[t][b] at columns (2t+b)*64, O_t at NQ*128 + t*128   (256 columns for NQ=1, 512 for NQ=2)
//   Tail  : tokens >= the end of the split inside the last tile are never valid data (page slack or
//           stale shared memory).  Their S columns are masked by selection; their V rows are zeroed
//           in shared memory by the MMA warp before P V, so no 0 x NaN can reach O.
//   Output: final bf16 rows (one split) or fp32 (m, l, o) partials for attn_combine_kernel.
#include <cuda_bf16.h>

#include "fcg_internal.h"

namespace fcg {
namespace {

constexpr int BM = 128;        // query rows per Q tile (UMMA M)
constexpr int BN = 64;         // cache tokens per K/V tile
constexpr int D = 128;
constexpr float RESCALE_TAU = 8.0f;   // log2 units: keep a stale row max while the new one is < 2^8 larger

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

// ---- mbarrier -----------------------------------------------------------------------------------
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
      "selp.u32 %0, 1, 0, p;\n\t"
      "}"
      : "=r"(ok)
      : "r"(bar), "r"(parity)
      : "memory");
  return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  while (!mbar_try_wait(bar, parity)) {
  }
}

__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// ---- TMA: one box of the 5-D pool tensor (D, P, Hkv, n_pages, L) -> shared memory ----------------
__device__ __forceinline__ void tma_load_5d(uint32_t dst, const TmaDesc *desc, uint32_t bar, int c0, int c1, int c2, int c3,
                                            int c4) {
  asm volatile(
      "cp.async.bulk.tensor.5d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5, %6}], [%7];" ::"r"(dst),
      "l"(reinterpret_cast<uint64_t>(desc)), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4), "r"(bar)
      : "memory");
}
__device__ __forceinline__ void tma_prefetch_desc(const TmaDesc *desc) {
  asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(desc)) : "memory");
}

// ---- tcgen05 --------------------------------------------------------------------------------------
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

template <int NCOLS>
__device__ __forceinline__ void tmem_alloc(uint32_t smem_dst) {
  asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_dst), "n"(NCOLS) : "memory");
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
template <int NCOLS>
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr) {
  asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "n"(NCOLS) : "memory");
}
__device__ __forceinline__ void umma_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
// D[tmem] (+)= A[smem] * B[smem]
__device__ __forceinline__ void umma_ss(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t"
      "}" ::"r"(d_tmem),
      "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate)
      : "memory");
}

// shared-memory matrix descriptor, 128B swizzle, version 1 (sm_100).  Offsets in bytes.
__device__ __forceinline__ uint64_t smem_desc(uint32_t addr, uint32_t lbo, uint32_t sbo) {
  const uint32_t lo = ((addr >> 4) & 0x3FFFu) | (((lbo >> 4) & 0x3FFFu) << 16);
  const uint32_t hi = ((sbo >> 4) & 0x3FFFu) | (1u << 14) | (2u << 29);
  return ((uint64_t)hi << 32) | lo;
}

// instruction descriptor, kind::f16: D fp32, A/B bf16, M = 128
constexpr uint32_t idesc_f16(int n, bool b_mn_major) {
  return (1u << 4) | (1u << 7) | (1u << 10) | ((b_mn_major ? 1u : 0u) << 16) | ((uint32_t)(n >> 3) << 17) |
         ((uint32_t)(BM >> 4) << 24);
}

#define TMEM_LD_32(taddr, r)                                                                                         \
  asm volatile(                                                                                                      \
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 "                                                                      \
      "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,"  \
      "%29,%30,%31}, [%32];"                                                                                         \
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),  \
        "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]),       \
        "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]),      \
        "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])                    \
      : "r"(taddr))

#define TMEM_ST_32(taddr, r)                                                                                         \
  asm volatile(                                                                                                      \
      "tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], "                                                                \
      "{%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29," \
      "%30,%31,%32};" ::"r"(taddr),                                                                                  \
      "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]), "r"(r[9]),  \
      "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15]), "r"(r[16]), "r"(r[17]), "r"(r[18]),    \
      "r"(r[19]), "r"(r[20]), "r"(r[21]), "r"(r[22]), "r"(r[23]), "r"(r[24]), "r"(r[25]), "r"(r[26]), "r"(r[27]),    \
      "r"(r[28]), "r"(r[29]), "r"(r[30]), "r"(r[31])                                                                 \
      : "memory")

__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
  __nv_bfloat162 r = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<uint32_t *>(&r);
}
__device__ __forceinline__ float ex2_approx(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

// ---- shared memory map -------------------------------------------------------------------------
constexpr int Q_TILE_B = BM * D * 2;          // two 64-column halves of [128][128 B]
constexpr int KV_TILE_B = BN * D * 2;         // two halves of [64][128 B]
constexpr int P_BYTES = BM * BN * 2;          // [128][128 B]

template <int NQ>
struct Cfg {
  static constexpr int KV_STAGES = NQ == 1 ? 4 : 3;
  static constexpr int N_SOFTMAX = NQ * BM;
  static constexpr int NTHREADS = N_SOFTMAX + 64;
  static constexpr int LOADER_WARP = 4 * NQ, MMA_WARP = 4 * NQ + 1;
  static constexpr int TMEM_COLS = NQ * 256;
  static constexpr int OFF_Q = 0;
  static constexpr int OFF_KV = OFF_Q + NQ * Q_TILE_B;               // stage s: K at +s*2*KV_TILE_B, V right after K
  static constexpr int OFF_P = OFF_KV + KV_STAGES * 2 * KV_TILE_B;   // P[t][b] at +(2t+b)*P_BYTES
  static constexpr int OFF_BAR = OFF_P + NQ * 2 * P_BYTES;
  // kv_full[ST], kv_empty[ST], s_full[NQ][2], p_full[NQ][2], pv_done[NQ][2], q_full
  static constexpr int N_BARS = 2 * KV_STAGES + 6 * NQ + 1;
  static constexpr int SMEM_BYTES = OFF_BAR + N_BARS * 8 + 16 + 1024;   // + tmem slot + alignment slack
};

template <int NQ>
__global__ void __launch_bounds__(Cfg<NQ>::NTHREADS, 1)
    attn_tc_kernel(const AttnParams p, const __grid_constant__ TmaDesc tm_k, const __grid_constant__ TmaDesc tm_v) {
  using C = Cfg<NQ>;
  constexpr int ST = C::KV_STAGES;
  extern __shared__ unsigned char smem_raw[];
  // 1024-byte alignment for the 128B-swizzle atoms
  unsigned char *smem = reinterpret_cast<unsigned char *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  const uint32_t sbase = smem_u32(smem);

  const int task_i = blockIdx.z % p.n_tasks;
  const int li = blockIdx.z / p.n_tasks;
  const AttnTaskDev tk = p.tasks[task_i];
  const int split = blockIdx.x % p.max_splits;
  const int rg = blockIdx.x / p.max_splits;
  const int G = p.group;
  const int R = tk.n * G;
  const int row0 = rg * (NQ * BM);                 // first query row of this CTA
  if (split >= tk.n_splits || row0 >= R) return;
  const int g = blockIdx.y;
  const int layer = p.layer_begin + li;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;

  const int t_begin = split * tk.split_len;
  const int t_end = min(tk.kv_len, t_begin + tk.split_len);
  const int32_t *pos = p.positions + tk.tok_off;
  const int cta_last = min(R, row0 + NQ * BM) - 1;
  const int cta_max_lim = min(pos[cta_last / G], t_end - 1);
  const int n_tiles = cta_max_lim >= t_begin ? (cta_max_lim - t_begin) / BN + 1 : 0;

  const uint32_t bar0 = sbase + C::OFF_BAR;
  auto kv_full = [&](int s) { return bar0 + 8 * s; };
  auto kv_empty = [&](int s) { return bar0 + 8 * (ST + s); };
  auto s_full = [&](int t, int b) { return bar0 + 8 * (2 * ST + 2 * t + b); };
  auto p_full = [&](int t, int b) { return bar0 + 8 * (2 * ST + 2 * NQ + 2 * t + b); };
  auto pv_done = [&](int t, int b) { return bar0 + 8 * (2 * ST + 4 * NQ + 2 * t + b); };
  const uint32_t q_full = bar0 + 8 * (2 * ST + 6 * NQ);
  const uint32_t tmem_slot = bar0 + 8 * C::N_BARS;
  volatile uint32_t *tmem_slot_ptr = reinterpret_cast<volatile uint32_t *>(smem + C::OFF_BAR + 8 * C::N_BARS);

  if (tid == 0) {
    for (int s = 0; s < ST; ++s) {
      mbar_init(kv_full(s), 1);
      mbar_init(kv_empty(s), 1);
    }
    for (int t = 0; t < NQ; ++t)
      for (int b = 0; b < 2; ++b) {
        mbar_init(s_full(t, b), 1);
        mbar_init(p_full(t, b), BM);
        mbar_init(pv_done(t, b), 1);
      }
    mbar_init(q_full, C::N_SOFTMAX);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == C::MMA_WARP) tmem_alloc<C::TMEM_COLS>(tmem_slot);
  if (warp == C::LOADER_WARP && lane == 0) {
    tma_prefetch_desc(&tm_k);
    tma_prefetch_desc(&tm_v);
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot_ptr;

  if (warp == C::LOADER_WARP) {
    // ======================================= loader ========================================
    // lane i of the warp owns page i of the tile: one page-table lookup, four box copies.
    const int P = p.page_size;
    const int ppt = BN / P;                         // pages per tile (P <= 64, power of two)
    const int32_t *table = p.tables + tk.table_off;
    auto page_of = [&](int j) -> int {
      const int tok = t_begin + j * BN + lane * P;
      return (j < n_tiles && lane < ppt && tok < t_end) ? __ldg(table + tok / P) : -1;
    };
    int page = page_of(0);
    for (int j = 0; j < n_tiles; ++j) {
      const int page_next = page_of(j + 1);         // issued before the wait: its latency hides behind it
      const int st = j % ST;
      if (j >= ST) mbar_wait(kv_empty(st), ((j / ST) - 1) & 1);
      const int ts = t_begin + j * BN;
      const int n_ok = min(ppt, (t_end - ts + P - 1) / P);
      if (lane == 0) mbar_arrive_expect_tx(kv_full(st), (uint32_t)(n_ok * P * (D * 2 * 2)));
      __syncwarp();
      if (page >= 0) {
        const uint32_t kdst = sbase + C::OFF_KV + st * (2 * KV_TILE_B) + lane * P * 128;
        const uint32_t vdst = kdst + KV_TILE_B;
        tma_load_5d(kdst, &tm_k, kv_full(st), 0, 0, g, page, layer);
        tma_load_5d(kdst + BN * 128, &tm_k, kv_full(st), 64, 0, g, page, layer);
        tma_load_5d(vdst, &tm_v, kv_full(st), 0, 0, g, page, layer);
        tma_load_5d(vdst + BN * 128, &tm_v, kv_full(st), 64, 0, g, page, layer);
      }
      page = page_next;
    }
  } else if (warp == C::MMA_WARP) {
    // ======================================= MMA issuer =====================================
    if (n_tiles > 0) {
      constexpr uint32_t IDESC_S = idesc_f16(BN, false);
      constexpr uint32_t IDESC_O = idesc_f16(D, true);
      mbar_wait(q_full, 0);
      auto issue_qk = [&](int j) {
        const int st = j % ST;
        mbar_wait(kv_full(st), (j / ST) & 1);
        const uint32_t kaddr = sbase + C::OFF_KV + st * (2 * KV_TILE_B);
        const int ts = t_begin + j * BN;
        if (ts + BN > t_end) {
          // ragged last tile: zero the V rows that hold no token of this split (whole warp)
          const int r0 = t_end - ts;
          unsigned char *vt = smem + C::OFF_KV + st * (2 * KV_TILE_B) + KV_TILE_B;
          for (int i = lane; i < (BN - r0) * 16; i += 32) {
            const int row = r0 + (i >> 4), c = i & 15;
            *reinterpret_cast<uint4 *>(vt + (c >> 3) * (BN * 128) + row * 128 + ((c & 7) << 4)) = make_uint4(0, 0, 0, 0);
          }
          fence_proxy_async();
          __syncwarp();
        }
        tc_fence_after();
        if (lane == 0) {
#pragma unroll
          for (int t = 0; t < NQ; ++t) {
#pragma unroll
            for (int k = 0; k < D / 16; ++k) {
              const uint64_t a = smem_desc(sbase + C::OFF_Q + t * Q_TILE_B + (k >> 2) * (BM * 128) + (k & 3) * 32, 16, 1024);
              const uint64_t b = smem_desc(kaddr + (k >> 2) * (BN * 128) + (k & 3) * 32, 16, 1024);
              umma_ss(tmem_base + (2 * t + (j & 1)) * BN, a, b, IDESC_S, k > 0);
            }
            umma_commit(s_full(t, j & 1));
          }
        }
        __syncwarp();
      };
      issue_qk(0);
      for (int j = 0; j < n_tiles; ++j) {
        if (j + 1 < n_tiles) issue_qk(j + 1);
        const int st = j % ST;
        const uint32_t vaddr = sbase + C::OFF_KV + st * (2 * KV_TILE_B) + KV_TILE_B;
#pragma unroll
        for (int t = 0; t < NQ; ++t) {
          mbar_wait(p_full(t, j & 1), (j >> 1) & 1);
          tc_fence_after();
          if (lane == 0) {
            const uint32_t paddr = sbase + C::OFF_P + (2 * t + (j & 1)) * P_BYTES;
            const uint32_t tmem_o = tmem_base + NQ * 128 + t * 128;
#pragma unroll
            for (int k = 0; k < BN / 16; ++k) {
              const uint64_t a = smem_desc(paddr + k * 32, 16, 1024);
              const uint64_t b = smem_desc(vaddr + k * 2048, BN * 128, 1024);   // MN-major: LBO = next 64-column half
              umma_ss(tmem_o, a, b, IDESC_O, (j > 0 || k > 0) ? 1u : 0u);
            }
            if (t == NQ - 1) umma_commit(kv_empty(st));
            umma_commit(pv_done(t, j & 1));
          }
          __syncwarp();
        }
      }
    }
  } else {
    // ======================================= softmax ========================================
    // Q tiles: rows r = row0 + row -> (token, head-in-group); rows past R are zero.  All softmax
    // threads copy cooperatively (coalesced 16-B chunks), then hand Q to the MMA thread.
    for (int i = 0; i < 16; ++i) {
      const int ci = tid + C::N_SOFTMAX * i;
      const int row = ci >> 4, c = ci & 15;
      const int r = row0 + row;
      uint4 val = make_uint4(0, 0, 0, 0);
      if (r < R) {
        const uint16_t *src = p.q + (((size_t)li * p.n_total + tk.tok_off + r / G) * p.n_q_heads + g * G + r % G) * D + c * 8;
        val = *reinterpret_cast<const uint4 *>(src);
      }
      const int rt = row & (BM - 1);
      const uint32_t dst = C::OFF_Q + (row >> 7) * Q_TILE_B + (c >> 3) * (BM * 128) + rt * 128 + (((c & 7) ^ (rt & 7)) << 4);
      *reinterpret_cast<uint4 *>(smem + dst) = val;
    }
    fence_proxy_async();
    mbar_arrive(q_full);

    const int qt = warp >> 2;                  // Q tile of this warp
    const int row = tid & (BM - 1);            // row in the tile == TMEM lane
    const int r = row0 + qt * BM + row;
    const bool valid = r < R;
    const int lim = valid ? min(pos[r / G], t_end - 1) : -1;
    const uint32_t lane_addr = ((uint32_t)((warp & 3) * 32) << 16);
    const uint32_t tmem_s = tmem_base + lane_addr + (2 * qt) * BN;
    const uint32_t tmem_o = tmem_base + lane_addr + NQ * 128 + qt * 128;
    const float sc = p.scale_log2;
    float m_ref = -INFINITY;                   // reference max used for exp2 (may lag the true max by < TAU)
    float l = 0.f;
    for (int j = 0; j < n_tiles; ++j) {
      const int ts = t_begin + j * BN;
      const int b = j & 1;
      mbar_wait(s_full(qt, b), (j >> 1) & 1);
      tc_fence_after();
      uint32_t sreg[2][32];
      TMEM_LD_32(tmem_s + b * BN, sreg[0]);
      TMEM_LD_32(tmem_s + b * BN + 32, sreg[1]);
      tmem_wait_ld();
      if (ts + BN - 1 > lim) {
#pragma unroll
        for (int h = 0; h < 2; ++h)
#pragma unroll
          for (int c = 0; c < 32; ++c)
            if (ts + h * 32 + c > lim) sreg[h][c] = 0xff800000u;   // -inf, by selection (S may be garbage there)
      }
      float mx4[4] = {-INFINITY, -INFINITY, -INFINITY, -INFINITY};
#pragma unroll
      for (int h = 0; h < 2; ++h)
#pragma unroll
        for (int c = 0; c < 32; ++c) mx4[c & 3] = fmaxf(mx4[c & 3], __uint_as_float(sreg[h][c]));
      const float mx = fmaxf(fmaxf(mx4[0], mx4[1]), fmaxf(mx4[2], mx4[3]));
      const float m_new = fmaxf(m_ref, mx * sc);
      // lazy rescale: move the reference only when it is too far behind
      float factor = 1.f;
      const bool bump = (m_new - m_ref > RESCALE_TAU) || (m_ref == -INFINITY && m_new != -INFINITY);
      if (bump) {
        factor = (m_ref == -INFINITY) ? 0.f : ex2_approx(m_ref - m_new);
        m_ref = m_new;
      }
      if (j > 0 && __any_sync(0xffffffffu, bump)) {
        // O holds tiles < j only once P V of tile j-1 has completed
        mbar_wait(pv_done(qt, (j - 1) & 1), ((j - 1) >> 1) & 1);
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
      // the P buffer of this parity was last read by P V of tile j-2
      if (j >= 2) mbar_wait(pv_done(qt, b), ((j - 2) >> 1) & 1);
      unsigned char *prow = smem + C::OFF_P + (2 * qt + b) * P_BYTES + row * 128;
      float sum4[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
      for (int c8 = 0; c8 < 8; ++c8) {
        float e[8];
#pragma unroll
        for (int c = 0; c < 8; ++c) {
          e[c] = ex2_approx(fmaf(__uint_as_float(sreg[c8 >> 2][(c8 & 3) * 8 + c]), sc, -mu));
          sum4[c & 3] += e[c];
        }
        uint4 v;
        v.x = pack_bf16(e[0], e[1]);
        v.y = pack_bf16(e[2], e[3]);
        v.z = pack_bf16(e[4], e[5]);
        v.w = pack_bf16(e[6], e[7]);
        *reinterpret_cast<uint4 *>(prow + ((c8 ^ (row & 7)) << 4)) = v;
      }
      l += (sum4[0] + sum4[1]) + (sum4[2] + sum4[3]);
      fence_proxy_async();
      tc_fence_before();
      mbar_arrive(p_full(qt, b));
    }

    // ---- epilogue: O / l -> bf16, or partials ---------------------------------------------
    if (n_tiles > 0) {
      mbar_wait(pv_done(qt, (n_tiles - 1) & 1), ((n_tiles - 1) >> 1) & 1);
      tc_fence_after();
    }
    const int i_tok = valid ? r / G : 0, hh = valid ? r % G : 0;
    const size_t out_row = ((size_t)li * p.n_total + tk.tok_off + i_tok) * p.n_q_heads + g * G + hh;
    const size_t prow_i = ((size_t)(li * p.max_splits + split) * p.n_total + tk.tok_off + i_tok) * p.n_q_heads + g * G + hh;
    const bool final_out = tk.n_splits == 1;
    const float inv = l > 0.f ? 1.f / l : 0.f;
#pragma unroll
    for (int ch = 0; ch < D / 32; ++ch) {
      uint32_t oreg[32];
      if (n_tiles > 0) {
        TMEM_LD_32(tmem_o + ch * 32, oreg);
        tmem_wait_ld();
      } else {
#pragma unroll
        for (int c = 0; c < 32; ++c) oreg[c] = 0u;
      }
      if (valid) {
        if (final_out) {
          uint16_t *dst = p.out + out_row * D + ch * 32;
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
          float *dst = p.part_o + prow_i * D + ch * 32;
#pragma unroll
          for (int c = 0; c < 32; c += 4)
            *reinterpret_cast<uint4 *>(dst + c) = make_uint4(oreg[c], oreg[c + 1], oreg[c + 2], oreg[c + 3]);
        }
      }
    }
    if (valid && !final_out) *reinterpret_cast<float2 *>(p.part_ml + prow_i * 2) = make_float2(m_ref, l);
  }

  tc_fence_before();
  __syncthreads();
  if (warp == C::MMA_WARP) {
    tc_fence_after();
    tmem_dealloc<C::TMEM_COLS>(tmem_base);
  }
}

template <int NQ>
cudaError_t launch_nq(const AttnParams &p, const TmaDesc &tk, const TmaDesc &tv, cudaStream_t stream) {
  using C = Cfg<NQ>;
  static bool configured = false;
  if (!configured) {
    cudaError_t e = cudaFuncSetAttribute(attn_tc_kernel<NQ>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_BYTES);
    if (e != cudaSuccess) return e;
    configured = true;
  }
  dim3 grid((unsigned)(p.max_splits * p.max_row_groups), (unsigned)p.n_kv_heads, (unsigned)(p.n_layers * p.n_tasks));
  attn_tc_kernel<NQ><<<grid, C::NTHREADS, C::SMEM_BYTES, stream>>>(p, tk, tv);
  return cudaGetLastError();
}

}  // namespace

// q_tiles = 128-row Q tiles per CTA (1 or 2); p.max_row_groups counts groups of q_tiles*128 rows.
cudaError_t launch_attn_tc(const AttnParams &p, int head_dim, int q_tiles, const TmaDesc *tm_k, const TmaDesc *tm_v,
                           cudaStream_t stream) {
  if (head_dim != 128 || !tm_k || !tm_v) return cudaErrorNotSupported;
  if (q_tiles == 1) return launch_nq<1>(p, *tm_k, *tm_v, stream);
  if (q_tiles == 2) return launch_nq<2>(p, *tm_k, *tm_v, stream);
  return cudaErrorInvalidValue;
}

}  // namespace fcg
