// S6: tensor-core patch attention on tcgen05 / TMEM (cache-patching, Eq. 6, PAPER.md:118-123, 718;
// DESIGN.md "Kernel S6").  Same result as the split-KV warp-MMA kernel, for R = n*G >= 64 query rows
// per kv head, where the two contractions Q K^T and P V are dense enough for the 5th-gen tensor cores.
//
//   CTA   = (KV split x 128-row group, kv head, layer x task); 288 threads, 1 CTA per SM
//   warps 0-3  softmax: thread == query row == TMEM lane.  S tile read with tcgen05.ld, online softmax
//              in the exp2 domain with a lazy (threshold 8) O rescale, P written as bf16 into a
//              128B-swizzled K-major shared-memory tile (the A operand of P V)
//   warps 4-7  loaders: cp.async 16 B (zero-fill past the end) through the page table into a 4-stage
//              ring of 128B-swizzled K and V tiles (64 tokens), handed to the MMA thread by mbarrier
//   warp  8    one thread issues tcgen05.mma (M=128, kind::f16, fp32 accumulate):
//              S[j&1] = Q K_j^T (N=64, K=128, both operands K-major)  and
//              O     += P_j V_j (N=128, K=64, V as an MN-major B operand), accumulators in TMEM
//   TMEM  = 256 columns: S0 [0,64), S1 [64,128), O [128,256)
//   QK^T of tile j+1 is issued before P V of tile j, so the softmax of tile j overlaps tensor work.
//   Output: final bf16 rows (one split) or fp32 (m, l, o) partials for attn_combine_kernel.
#include <cuda_bf16.h>

#include "fcg_internal.h"

namespace fcg {
namespace {

constexpr int BM = 128;        // query rows per CTA (UMMA M)
constexpr int BN = 64;         // cache tokens per tile
constexpr int KV_STAGES = 4;
constexpr int LOOKAHEAD = KV_STAGES - 1;
constexpr int N_SOFTMAX = 128, N_LOADER = 128;
constexpr int NTHREADS = N_SOFTMAX + N_LOADER + 32;
constexpr float RESCALE_TAU = 8.0f;   // log2 units: keep a stale row max while the new one is < 2^8 larger

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

// ---- mbarrier -----------------------------------------------------------------------------------
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
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

// ---- cp.async -------------------------------------------------------------------------------------
__device__ __forceinline__ void cp_async_16_zfill(uint32_t dst, const void *src, int src_bytes) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
  asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// ---- tcgen05 --------------------------------------------------------------------------------------
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

__device__ __forceinline__ void tmem_alloc(uint32_t smem_dst, uint32_t ncols) {
  asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_dst), "r"(ncols) : "memory");
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr, uint32_t ncols) {
  asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols) : "memory");
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

// ---- shared memory map (D = 128) ---------------------------------------------------------------
constexpr int D = 128;
constexpr int Q_BYTES = BM * D * 2;           // two 64-column halves of [128][128 B]
constexpr int KV_TILE_B = BN * D * 2;         // two halves of [64][128 B]
constexpr int P_BYTES = BM * BN * 2;          // [128][128 B]
constexpr int OFF_Q = 0;
constexpr int OFF_KV = OFF_Q + Q_BYTES;                           // stage s: K at +s*2*KV_TILE_B, V right after K
constexpr int OFF_P = OFF_KV + KV_STAGES * 2 * KV_TILE_B;
constexpr int OFF_BAR = OFF_P + 2 * P_BYTES;
constexpr int N_BARS = 2 * KV_STAGES + 2 + 2 + 2 + 1;             // kv_full, kv_empty, s_full[2], p_full[2], pv_done[2], q_full
constexpr int SMEM_BYTES = OFF_BAR + N_BARS * 8 + 16 + 1024;      // + tmem slot + alignment slack

__global__ void __launch_bounds__(NTHREADS, 1) attn_tc_kernel(const AttnParams p) {
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
  if (split >= tk.n_splits || rg * BM >= R) return;
  const int g = blockIdx.y;
  const int layer = p.layer_begin + li;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;

  const int t_begin = split * tk.split_len;
  const int t_end = min(tk.kv_len, t_begin + tk.split_len);
  const int32_t *pos = p.positions + tk.tok_off;
  const int cta_last = min(R, rg * BM + BM) - 1;
  const int cta_max_lim = min(pos[cta_last / G], t_end - 1);
  const int n_tiles = cta_max_lim >= t_begin ? (cta_max_lim - t_begin) / BN + 1 : 0;

  const uint32_t bar0 = sbase + OFF_BAR;
  auto kv_full = [&](int s) { return bar0 + 8 * s; };
  auto kv_empty = [&](int s) { return bar0 + 8 * (KV_STAGES + s); };
  auto s_full = [&](int b) { return bar0 + 8 * (2 * KV_STAGES + b); };
  auto p_full = [&](int b) { return bar0 + 8 * (2 * KV_STAGES + 2 + b); };
  auto pv_done = [&](int b) { return bar0 + 8 * (2 * KV_STAGES + 4 + b); };
  const uint32_t q_full = bar0 + 8 * (2 * KV_STAGES + 6);
  const uint32_t tmem_slot = bar0 + 8 * N_BARS;
  volatile uint32_t *tmem_slot_ptr = reinterpret_cast<volatile uint32_t *>(smem + OFF_BAR + 8 * N_BARS);

  if (tid == 0) {
    for (int s = 0; s < KV_STAGES; ++s) {
      mbar_init(kv_full(s), N_LOADER);
      mbar_init(kv_empty(s), 1);
    }
    for (int b = 0; b < 2; ++b) {
      mbar_init(s_full(b), 1);
      mbar_init(p_full(b), N_SOFTMAX);
      mbar_init(pv_done(b), 1);
    }
    mbar_init(q_full, N_LOADER);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 8) tmem_alloc(tmem_slot, 256);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot_ptr;

  if (warp >= 4 && warp < 8) {
    // ======================================= loaders =======================================
    const int lt = tid - N_SOFTMAX;
    // Q tile: rows r = rg*BM + row -> (token, head-in-group); rows past R are zero
    for (int i = 0; i < (BM * 16) / N_LOADER; ++i) {
      const int ci = lt + N_LOADER * i;
      const int row = ci >> 4, c = ci & 15;
      const int r = rg * BM + row;
      uint4 val = make_uint4(0, 0, 0, 0);
      if (r < R) {
        const uint16_t *src = p.q + (((size_t)li * p.n_total + tk.tok_off + r / G) * p.n_q_heads + g * G + r % G) * D + c * 8;
        val = *reinterpret_cast<const uint4 *>(src);
      }
      const uint32_t dst = OFF_Q + (c >> 3) * (BM * 128) + row * 128 + (((c & 7) ^ (row & 7)) << 4);
      *reinterpret_cast<uint4 *>(smem + dst) = val;
    }
    fence_proxy_async();
    mbar_arrive(q_full);

    const int32_t *table = p.tables + tk.table_off;
    const size_t head_stride = (size_t)p.page_size * D;
    const size_t page_stride = head_stride * p.n_kv_heads;
    const size_t layer_base = ((size_t)layer * p.n_pages) * page_stride + (size_t)g * head_stride;
    for (int j = 0; j < n_tiles + LOOKAHEAD; ++j) {
      // Hand tile j-LOOKAHEAD over BEFORE blocking on a free stage for tile j: the stage of tile j is
      // released by P V of tile j-KV_STAGES, which the MMA thread issues only after Q K^T of tile
      // j-KV_STAGES+1 = j-LOOKAHEAD -- the tile signalled here.  (The other order deadlocks as soon as
      // a CTA has more than KV_STAGES tiles.)
      if (j >= LOOKAHEAD) {
        cp_async_wait<LOOKAHEAD - 1>();
        fence_proxy_async();
        mbar_arrive(kv_full((j - LOOKAHEAD) % KV_STAGES));
      }
      if (j < n_tiles) {
        const int st = j % KV_STAGES;
        if (j >= KV_STAGES) mbar_wait(kv_empty(st), ((j / KV_STAGES) - 1) & 1);
        const int ts = t_begin + j * BN;
        const uint32_t kdst = sbase + OFF_KV + st * (2 * KV_TILE_B);
        const uint32_t vdst = kdst + KV_TILE_B;
#pragma unroll
        for (int i = 0; i < (BN * 16) / N_LOADER; ++i) {
          const int ci = lt + N_LOADER * i;
          const int t = ci >> 4, c = ci & 15;
          const int tok = ts + t;
          const bool ok = tok < t_end;
          size_t off = 0;
          if (ok) {
            const int page = table[tok / p.page_size];
            off = layer_base + (size_t)page * page_stride + (size_t)(tok % p.page_size) * D + c * 8;
          }
          const uint32_t so = (c >> 3) * (BN * 128) + t * 128 + (((c & 7) ^ (t & 7)) << 4);
          cp_async_16_zfill(kdst + so, p.k_pool + off, ok ? 16 : 0);
          cp_async_16_zfill(vdst + so, p.v_pool + off, ok ? 16 : 0);
        }
      }
      cp_async_commit();
    }
  } else if (warp == 8) {
    // ======================================= MMA issuer =====================================
    if (lane == 0 && n_tiles > 0) {
      constexpr uint32_t IDESC_S = idesc_f16(BN, false);
      constexpr uint32_t IDESC_O = idesc_f16(D, true);
      const uint32_t tmem_o = tmem_base + 128;
      mbar_wait(q_full, 0);
      auto issue_qk = [&](int j) {
        const int st = j % KV_STAGES;
        mbar_wait(kv_full(st), (j / KV_STAGES) & 1);
        tc_fence_after();
        const uint32_t kaddr = sbase + OFF_KV + st * (2 * KV_TILE_B);
#pragma unroll
        for (int k = 0; k < D / 16; ++k) {
          const uint64_t a = smem_desc(sbase + OFF_Q + (k >> 2) * (BM * 128) + (k & 3) * 32, 16, 1024);
          const uint64_t b = smem_desc(kaddr + (k >> 2) * (BN * 128) + (k & 3) * 32, 16, 1024);
          umma_ss(tmem_base + (j & 1) * BN, a, b, IDESC_S, k > 0);
        }
        umma_commit(s_full(j & 1));
      };
      issue_qk(0);
      for (int j = 0; j < n_tiles; ++j) {
        if (j + 1 < n_tiles) issue_qk(j + 1);
        mbar_wait(p_full(j & 1), (j >> 1) & 1);
        tc_fence_after();
        const int st = j % KV_STAGES;
        const uint32_t vaddr = sbase + OFF_KV + st * (2 * KV_TILE_B) + KV_TILE_B;
        const uint32_t paddr = sbase + OFF_P + (j & 1) * P_BYTES;
#pragma unroll
        for (int k = 0; k < BN / 16; ++k) {
          const uint64_t a = smem_desc(paddr + k * 32, 16, 1024);
          const uint64_t b = smem_desc(vaddr + k * 2048, BN * 128, 1024);   // MN-major: LBO = next 64-column half
          umma_ss(tmem_o, a, b, IDESC_O, (j > 0 || k > 0) ? 1u : 0u);
        }
        umma_commit(kv_empty(st));
        umma_commit(pv_done(j & 1));
      }
    }
  } else {
    // ======================================= softmax ========================================
    const int row = tid;                       // == TMEM lane
    const int r = rg * BM + row;
    const bool valid = r < R;
    const int lim = valid ? min(pos[r / G], t_end - 1) : -1;
    const uint32_t lane_addr = ((uint32_t)(warp * 32) << 16);
    const float sc = p.scale_log2;
    float m_ref = -INFINITY;                   // reference max used for exp2 (may lag the true max by < TAU)
    float l = 0.f;
    for (int j = 0; j < n_tiles; ++j) {
      const int ts = t_begin + j * BN;
      mbar_wait(s_full(j & 1), (j >> 1) & 1);
      tc_fence_after();
      uint32_t sreg[2][32];
      TMEM_LD_32(tmem_base + lane_addr + (j & 1) * BN, sreg[0]);
      TMEM_LD_32(tmem_base + lane_addr + (j & 1) * BN + 32, sreg[1]);
      tmem_wait_ld();
      float mx = -INFINITY;
      const bool need_mask = ts + BN - 1 > lim;
#pragma unroll
      for (int h = 0; h < 2; ++h)
#pragma unroll
        for (int c = 0; c < 32; ++c) {
          float s = __uint_as_float(sreg[h][c]);
          if (need_mask && ts + h * 32 + c > lim) s = -INFINITY;
          sreg[h][c] = __float_as_uint(s);
          mx = fmaxf(mx, s);
        }
      const float m_new = fmaxf(m_ref, mx * sc);
      // lazy rescale: move the reference only when it is too far behind
      float factor = 1.f;
      bool bump = (m_new - m_ref > RESCALE_TAU) || (m_ref == -INFINITY && m_new != -INFINITY);
      if (bump) {
        factor = (m_ref == -INFINITY) ? 0.f : exp2f(m_ref - m_new);
        m_ref = m_new;
      }
      const bool warp_bump = __any_sync(0xffffffffu, bump) && j > 0;
      if (warp_bump) {
        // O holds tiles < j only once P V of tile j-1 has completed
        mbar_wait(pv_done((j - 1) & 1), ((j - 1) >> 1) & 1);
        tc_fence_after();
#pragma unroll
        for (int ch = 0; ch < D / 32; ++ch) {
          uint32_t oreg[32];
          TMEM_LD_32(tmem_base + lane_addr + 128 + ch * 32, oreg);
          tmem_wait_ld();
#pragma unroll
          for (int c = 0; c < 32; ++c) oreg[c] = __float_as_uint(__uint_as_float(oreg[c]) * factor);
          TMEM_ST_32(tmem_base + lane_addr + 128 + ch * 32, oreg);
        }
        tmem_wait_st();
      }
      l *= factor;
      const float mu = m_ref == -INFINITY ? 0.f : m_ref;
      // the P buffer of this parity was last read by P V of tile j-2
      if (j >= 2) mbar_wait(pv_done(j & 1), ((j - 2) >> 1) & 1);
      unsigned char *prow = smem + OFF_P + (j & 1) * P_BYTES + row * 128;
      float sum = 0.f;
#pragma unroll
      for (int c8 = 0; c8 < 8; ++c8) {
        float e[8];
#pragma unroll
        for (int c = 0; c < 8; ++c) {
          e[c] = exp2f(fmaf(__uint_as_float(sreg[c8 >> 2][(c8 & 3) * 8 + c]), sc, -mu));
          sum += e[c];
        }
        uint4 v;
        v.x = pack_bf16(e[0], e[1]);
        v.y = pack_bf16(e[2], e[3]);
        v.z = pack_bf16(e[4], e[5]);
        v.w = pack_bf16(e[6], e[7]);
        *reinterpret_cast<uint4 *>(prow + ((c8 ^ (row & 7)) << 4)) = v;
      }
      l += sum;
      fence_proxy_async();
      tc_fence_before();
      mbar_arrive(p_full(j & 1));
    }

    // ---- epilogue: O / l -> bf16, or partials ---------------------------------------------
    if (n_tiles > 0) {
      mbar_wait(pv_done((n_tiles - 1) & 1), ((n_tiles - 1) >> 1) & 1);
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
        TMEM_LD_32(tmem_base + lane_addr + 128 + ch * 32, oreg);
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
  if (warp == 8) {
    tc_fence_after();
    tmem_dealloc(tmem_base, 256);
  }
}

}  // namespace

cudaError_t launch_attn_tc(const AttnParams &p, int head_dim, cudaStream_t stream) {
  if (head_dim != 128) return cudaErrorNotSupported;
  static bool configured = false;
  if (!configured) {
    cudaError_t e = cudaFuncSetAttribute(attn_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
    if (e != cudaSuccess) return e;
    configured = true;
  }
  dim3 grid((unsigned)(p.max_splits * p.max_row_groups), (unsigned)p.n_kv_heads, (unsigned)(p.n_layers * p.n_tasks));
  attn_tc_kernel<<<grid, NTHREADS, SMEM_BYTES, stream>>>(p);
  return cudaGetLastError();
}

}  // namespace fcg
