// S5: short-patch causal attention over the stitched paged cache (cache-patching, Eq. 6,
// PAPER.md:118-123, 718).  Split-KV, bandwidth-bound: every visible K/V byte is
// streamed once per kv head; the R = n*G query rows that share a kv head ride along in registers.
//
//   grid  = (split x row-group, kv head, layer x task), 128 threads = 4 warps, 2 CTAs per SM
//   tile  = 64 cache tokens of K and V, cp.async (16 B, zero-fill past the end) through the page table
//           into a 3-stage XOR-swizzled shared-memory ring
//   math  = mma.sync m16n8k16 bf16 (fp32 accumulate) for Q K^T and P V, warp-shuffle online softmax
//           in the exp2 domain; rows are (token, q-head-in-group) pairs, 16 per warp
//   MB    = 16-row blocks per CTA (1, 2 or 4).  With MB < 4 the 4/MB spare warps split each tile's
//           tokens among themselves (an in-CTA split-KV), merged through shared memory at the end.
//   out   = final bf16 rows if the task has one split, else fp32 (m, l, o) partials merged by
//           attn_combine_kernel with a log-sum-exp.
#include <cuda_bf16.h>

#include "fcg_internal.h"

namespace fcg {
namespace {

constexpr int BN = 64;       // cache tokens per tile
constexpr int STAGES = 3;
constexpr int NTHREADS = 128;

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void cp_async_16_zfill(uint32_t dst, const void *src, int src_bytes) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
  asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory");
}

__device__ __forceinline__ void ldmatrix_x4(uint32_t &r0, uint32_t &r1, uint32_t &r2, uint32_t &r3, uint32_t addr) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];"
               : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3)
               : "r"(addr));
}
__device__ __forceinline__ void ldmatrix_x4_trans(uint32_t &r0, uint32_t &r1, uint32_t &r2, uint32_t &r3,
                                                  uint32_t addr) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];"
               : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3)
               : "r"(addr));
}
__device__ __forceinline__ void mma_bf16_16816(float (&c)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
  asm volatile(
      "mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
      : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
      : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
  __nv_bfloat162 r = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<uint32_t *>(&r);
}

template <int D, int MB>
__global__ void __launch_bounds__(NTHREADS, 2) attn_split_kernel(const AttnParams p) {
  constexpr int NS = 4 / MB;             // token slices per tile
  constexpr int SL = BN / NS;            // tokens per slice
  constexpr int NT_S = SL / 8;           // score n-tiles per warp
  constexpr int KS_P = SL / 16;          // k-steps of P V per warp
  constexpr int BM = 16 * MB;
  constexpr int ROW_B = D * 2;           // bytes per K/V row
  constexpr int CPR = D / 8;             // 16-byte chunks per row
  constexpr int TILE_B = BN * ROW_B;
  constexpr int ROWS_PER_PASS = NTHREADS / CPR;
  constexpr int PASSES = BN / ROWS_PER_PASS;
  constexpr int OPAD = D + 8;            // fp32 row stride of the merge buffer

  extern __shared__ __align__(128) unsigned char smem[];

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
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int rb = warp % MB, sl = warp / MB;
  const int so = sl * SL;

  const int t_begin = split * tk.split_len;
  const int t_end = min(tk.kv_len, t_begin + tk.split_len);
  const int32_t *pos = p.positions + tk.tok_off;

  // rows are r = i*G + hh (token-major), so limits are non-decreasing in r
  const int cta_last = min(R, rg * BM + BM) - 1;
  const int cta_max_lim = min(pos[cta_last / G], t_end - 1);
  const int n_tiles = cta_max_lim >= t_begin ? (cta_max_lim - t_begin) / BN + 1 : 0;

  const int wb_first = rg * BM + rb * 16;
  const bool warp_has_rows = wb_first < R;
  int wmax_lim = -1, wmin_lim = -1;
  if (warp_has_rows) {
    wmax_lim = min(pos[(min(R, wb_first + 16) - 1) / G], t_end - 1);
    wmin_lim = (wb_first + 16 <= R) ? min(pos[wb_first / G], t_end - 1) : -1;
  }
  const int r0 = wb_first + (lane >> 2), r1 = r0 + 8;
  const int lim0 = r0 < R ? min(pos[r0 / G], t_end - 1) : -1;
  const int lim1 = r1 < R ? min(pos[r1 / G], t_end - 1) : -1;

  // ---- Q fragments (A operand), straight from global ------------------------------------------
  uint32_t qf[D / 16][4];
  {
    const uint16_t *q0 = p.q + (((size_t)li * p.n_total + tk.tok_off + (r0 < R ? r0 / G : 0)) * p.n_q_heads + g * G +
                                (r0 < R ? r0 % G : 0)) * D;
    const uint16_t *q1 = p.q + (((size_t)li * p.n_total + tk.tok_off + (r1 < R ? r1 / G : 0)) * p.n_q_heads + g * G +
                                (r1 < R ? r1 % G : 0)) * D;
    const int c = 2 * (lane & 3);
#pragma unroll
    for (int ks = 0; ks < D / 16; ++ks) {
      qf[ks][0] = r0 < R ? *reinterpret_cast<const uint32_t *>(q0 + ks * 16 + c) : 0u;
      qf[ks][1] = r1 < R ? *reinterpret_cast<const uint32_t *>(q1 + ks * 16 + c) : 0u;
      qf[ks][2] = r0 < R ? *reinterpret_cast<const uint32_t *>(q0 + ks * 16 + 8 + c) : 0u;
      qf[ks][3] = r1 < R ? *reinterpret_cast<const uint32_t *>(q1 + ks * 16 + 8 + c) : 0u;
    }
  }

  // ---- tile loader ---------------------------------------------------------------------------------
  const int32_t *table = p.tables + tk.table_off;
  const size_t head_stride = (size_t)p.page_size * D;                       // elements
  const size_t page_stride = head_stride * p.n_kv_heads;
  const size_t layer_base = ((size_t)layer * p.n_pages) * page_stride + (size_t)g * head_stride;
  const int lc = tid % CPR, lr = tid / CPR;
  const uint32_t smem_base = smem_u32(smem);

  auto load_tile = [&](int tile, int stage) {
    const int ts = t_begin + tile * BN;
    const uint32_t kdst = smem_base + stage * (2 * TILE_B);
    const uint32_t vdst = kdst + TILE_B;
#pragma unroll
    for (int i = 0; i < PASSES; ++i) {
      const int rr = lr + i * ROWS_PER_PASS;
      const int tok = ts + rr;
      const bool ok = tok < t_end;
      size_t off = 0;
      if (ok) {
        const int page = table[tok / p.page_size];
        off = layer_base + (size_t)page * page_stride + (size_t)(tok % p.page_size) * D + lc * 8;
      }
      const uint32_t so_b = rr * ROW_B + ((lc ^ (rr & 7)) << 4);
      cp_async_16_zfill(kdst + so_b, p.k_pool + off, ok ? 16 : 0);
      cp_async_16_zfill(vdst + so_b, p.v_pool + off, ok ? 16 : 0);
    }
  };

  // ---- state ---------------------------------------------------------------------------------------
  float o[D / 8][4];
#pragma unroll
  for (int i = 0; i < D / 8; ++i) o[i][0] = o[i][1] = o[i][2] = o[i][3] = 0.f;
  float m0 = -INFINITY, m1 = -INFINITY, l0 = 0.f, l1 = 0.f;
  const float sc = p.scale_log2;

#pragma unroll
  for (int s = 0; s < STAGES - 1; ++s) {
    if (s < n_tiles) load_tile(s, s);
    cp_async_commit();
  }

  for (int tile = 0; tile < n_tiles; ++tile) {
    cp_async_wait<STAGES - 2>();
    __syncthreads();
    if (tile + STAGES - 1 < n_tiles) load_tile(tile + STAGES - 1, (tile + STAGES - 1) % STAGES);
    cp_async_commit();

    const int ts = t_begin + tile * BN + so;       // first token of this warp's slice
    if (!warp_has_rows || ts > wmax_lim) continue;  // nothing visible to this warp's rows
    const uint32_t kbase = smem_base + (tile % STAGES) * (2 * TILE_B);
    const uint32_t vbase = kbase + TILE_B;

    float s[NT_S][4];
#pragma unroll
    for (int nt = 0; nt < NT_S; ++nt) s[nt][0] = s[nt][1] = s[nt][2] = s[nt][3] = 0.f;
#pragma unroll
    for (int ks2 = 0; ks2 < D / 32; ++ks2) {
#pragma unroll
      for (int nt = 0; nt < NT_S; ++nt) {
        const int row = so + nt * 8 + (lane & 7);
        const int cidx = ks2 * 4 + (lane >> 3);
        uint32_t b0, b1, b2, b3;
        ldmatrix_x4(b0, b1, b2, b3, kbase + row * ROW_B + ((cidx ^ (row & 7)) << 4));
        mma_bf16_16816(s[nt], qf[2 * ks2], b0, b1);
        mma_bf16_16816(s[nt], qf[2 * ks2 + 1], b2, b3);
      }
    }

    if (ts + SL - 1 > wmin_lim) {   // causal / end-of-range mask
#pragma unroll
      for (int nt = 0; nt < NT_S; ++nt) {
        const int tok = ts + nt * 8 + 2 * (lane & 3);
        if (tok > lim0) s[nt][0] = -INFINITY;
        if (tok + 1 > lim0) s[nt][1] = -INFINITY;
        if (tok > lim1) s[nt][2] = -INFINITY;
        if (tok + 1 > lim1) s[nt][3] = -INFINITY;
      }
    }

    float mx0 = -INFINITY, mx1 = -INFINITY;
#pragma unroll
    for (int nt = 0; nt < NT_S; ++nt) {
      mx0 = fmaxf(mx0, fmaxf(s[nt][0], s[nt][1]));
      mx1 = fmaxf(mx1, fmaxf(s[nt][2], s[nt][3]));
    }
    mx0 = fmaxf(mx0, __shfl_xor_sync(0xffffffffu, mx0, 1));
    mx0 = fmaxf(mx0, __shfl_xor_sync(0xffffffffu, mx0, 2));
    mx1 = fmaxf(mx1, __shfl_xor_sync(0xffffffffu, mx1, 1));
    mx1 = fmaxf(mx1, __shfl_xor_sync(0xffffffffu, mx1, 2));
    const float mn0 = fmaxf(m0, mx0 * sc), mn1 = fmaxf(m1, mx1 * sc);
    const float mu0 = mn0 == -INFINITY ? 0.f : mn0, mu1 = mn1 == -INFINITY ? 0.f : mn1;
    const float c0 = exp2f(m0 - mu0), c1 = exp2f(m1 - mu1);
    m0 = mn0;
    m1 = mn1;
    float sum0 = 0.f, sum1 = 0.f;
#pragma unroll
    for (int nt = 0; nt < NT_S; ++nt) {
      s[nt][0] = exp2f(fmaf(s[nt][0], sc, -mu0));
      s[nt][1] = exp2f(fmaf(s[nt][1], sc, -mu0));
      s[nt][2] = exp2f(fmaf(s[nt][2], sc, -mu1));
      s[nt][3] = exp2f(fmaf(s[nt][3], sc, -mu1));
      sum0 += s[nt][0] + s[nt][1];
      sum1 += s[nt][2] + s[nt][3];
    }
    l0 = l0 * c0 + sum0;
    l1 = l1 * c1 + sum1;
#pragma unroll
    for (int i = 0; i < D / 8; ++i) {
      o[i][0] *= c0;
      o[i][1] *= c0;
      o[i][2] *= c1;
      o[i][3] *= c1;
    }

#pragma unroll
    for (int kk = 0; kk < KS_P; ++kk) {
      uint32_t a[4];
      a[0] = pack_bf16(s[2 * kk][0], s[2 * kk][1]);
      a[1] = pack_bf16(s[2 * kk][2], s[2 * kk][3]);
      a[2] = pack_bf16(s[2 * kk + 1][0], s[2 * kk + 1][1]);
      a[3] = pack_bf16(s[2 * kk + 1][2], s[2 * kk + 1][3]);
      const int m = lane >> 3;
      const int trow = so + kk * 16 + (m & 1) * 8 + (lane & 7);
#pragma unroll
      for (int np = 0; np < D / 16; ++np) {
        const int cidx = np * 2 + (m >> 1);
        uint32_t b0, b1, b2, b3;
        ldmatrix_x4_trans(b0, b1, b2, b3, vbase + trow * ROW_B + ((cidx ^ (trow & 7)) << 4));
        mma_bf16_16816(o[2 * np], a, b0, b1);
        mma_bf16_16816(o[2 * np + 1], a, b2, b3);
      }
    }
  }

  cp_async_wait<0>();
  __syncthreads();   // the ring is free: reuse it as the merge buffer

  l0 += __shfl_xor_sync(0xffffffffu, l0, 1);
  l0 += __shfl_xor_sync(0xffffffffu, l0, 2);
  l1 += __shfl_xor_sync(0xffffffffu, l1, 1);
  l1 += __shfl_xor_sync(0xffffffffu, l1, 2);

  float *so_buf = reinterpret_cast<float *>(smem);          // [4 warps][16][OPAD]
  float *sm_buf = so_buf + 4 * 16 * OPAD;                   // [4][16] m
  float *sl_buf = sm_buf + 4 * 16;                          // [4][16] l
  {
    float *wo = so_buf + warp * 16 * OPAD;
    const int rr = lane >> 2, cc = 2 * (lane & 3);
#pragma unroll
    for (int i = 0; i < D / 8; ++i) {
      *reinterpret_cast<float2 *>(wo + rr * OPAD + i * 8 + cc) = make_float2(o[i][0], o[i][1]);
      *reinterpret_cast<float2 *>(wo + (rr + 8) * OPAD + i * 8 + cc) = make_float2(o[i][2], o[i][3]);
    }
    if ((lane & 3) == 0) {
      sm_buf[warp * 16 + rr] = m0;
      sm_buf[warp * 16 + rr + 8] = m1;
      sl_buf[warp * 16 + rr] = l0;
      sl_buf[warp * 16 + rr + 8] = l1;
    }
  }
  __syncthreads();

  // ---- row owners: merge the NS slices and write ----------------------------------------------
  constexpr int TPR = NTHREADS / BM;     // threads per row
  constexpr int CPT = D / TPR;           // columns per thread
  const int row = tid / TPR;
  const int r = rg * BM + row;
  if (r >= R) return;
  const int cb = (tid % TPR) * CPT;
  const int orb = row / 16, orr = row % 16;
  float M = -INFINITY;
#pragma unroll
  for (int s2 = 0; s2 < NS; ++s2) M = fmaxf(M, sm_buf[(orb + MB * s2) * 16 + orr]);
  const float Mu = M == -INFINITY ? 0.f : M;
  float L = 0.f;
  float w[NS];
#pragma unroll
  for (int s2 = 0; s2 < NS; ++s2) {
    w[s2] = exp2f(sm_buf[(orb + MB * s2) * 16 + orr] - Mu);
    L += w[s2] * sl_buf[(orb + MB * s2) * 16 + orr];
  }
  const int i_tok = r / G, hh = r % G;
  const size_t out_row = ((size_t)li * p.n_total + tk.tok_off + i_tok) * p.n_q_heads + g * G + hh;
  if (tk.n_splits == 1) {
    const float inv = L > 0.f ? 1.f / L : 0.f;
    uint16_t *dst = p.out + out_row * D + cb;
#pragma unroll
    for (int c = 0; c < CPT; c += 2) {
      float a0 = 0.f, a1 = 0.f;
#pragma unroll
      for (int s2 = 0; s2 < NS; ++s2) {
        const float *src = so_buf + ((orb + MB * s2) * 16 + orr) * OPAD + cb + c;
        a0 += w[s2] * src[0];
        a1 += w[s2] * src[1];
      }
      *reinterpret_cast<uint32_t *>(dst + c) = pack_bf16(a0 * inv, a1 * inv);
    }
  } else {
    const size_t prow = ((size_t)(li * p.max_splits + split) * p.n_total + tk.tok_off + i_tok) * p.n_q_heads + g * G + hh;
    float *dst = p.part_o + prow * D + cb;
#pragma unroll
    for (int c = 0; c < CPT; c += 2) {
      float a0 = 0.f, a1 = 0.f;
#pragma unroll
      for (int s2 = 0; s2 < NS; ++s2) {
        const float *src = so_buf + ((orb + MB * s2) * 16 + orr) * OPAD + cb + c;
        a0 += w[s2] * src[0];
        a1 += w[s2] * src[1];
      }
      *reinterpret_cast<float2 *>(dst + c) = make_float2(a0, a1);
    }
    if (tid % TPR == 0) *reinterpret_cast<float2 *>(p.part_ml + prow * 2) = make_float2(M, L);
  }
}

// one warp per (layer, token, q head) row: log-sum-exp merge of the splits.  The (m, l) pairs of the splits are read by
// the lanes in parallel (split s in lane s % 32) and reduced with shuffles; the partial rows are then accumulated four
// splits at a time with all their loads in flight.  (The first version walked the splits one by one, twice, and took 11 us
// for a single layer of C3 -- 4096 rows x 9 splits, all of it L2 latency.)
struct CombineRow {
  size_t rowi, prow0, stride;     // output row; partial row of split 0; partial-row stride between splits
  int ns;
  float w0, w1, inv;              // this lane's weights for the splits `lane` and `lane + 32`; 1 / L
};

__device__ __forceinline__ bool combine_prologue(const AttnParams &p, CombineRow &c) {
  const size_t n_rows = (size_t)p.n_layers * p.n_total * p.n_q_heads;
  c.rowi = (size_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (c.rowi >= n_rows) return false;
  const int lane = threadIdx.x & 31;
  const int h = (int)(c.rowi % p.n_q_heads);
  const size_t lt = c.rowi / p.n_q_heads;
  const int tok = (int)(lt % p.n_total);
  const int li = (int)(lt / p.n_total);
  c.ns = p.tok_splits[tok];
  if (c.ns <= 1) return false;    // the attention kernel already wrote the final row
  c.stride = (size_t)p.n_total * p.n_q_heads;
  c.prow0 = ((size_t)li * p.max_splits * p.n_total + tok) * p.n_q_heads + h;
  float2 a = make_float2(-INFINITY, 0.f), b = make_float2(-INFINITY, 0.f);
  if (lane < c.ns) a = *reinterpret_cast<const float2 *>(p.part_ml + (c.prow0 + (size_t)lane * c.stride) * 2);
  if (lane + 32 < c.ns) b = *reinterpret_cast<const float2 *>(p.part_ml + (c.prow0 + (size_t)(lane + 32) * c.stride) * 2);
  float M = fmaxf(a.x, b.x);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) M = fmaxf(M, __shfl_xor_sync(0xffffffffu, M, o));
  const float Mu = M == -INFINITY ? 0.f : M;
  c.w0 = lane < c.ns ? exp2f(a.x - Mu) : 0.f;
  c.w1 = lane + 32 < c.ns ? exp2f(b.x - Mu) : 0.f;
  float L = c.w0 * a.y + c.w1 * b.y;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) L += __shfl_xor_sync(0xffffffffu, L, o);
  c.inv = L > 0.f ? 1.f / L : 0.f;
  return true;
}

template <int D>
__global__ void __launch_bounds__(256) attn_combine_kernel(const AttnParams p) {
  asm volatile("griddepcontrol.wait;" ::: "memory");   // pre-launched behind the attention kernel (no-op otherwise)
  constexpr int CPL = D / 32;                          // consecutive floats per lane: 2, 4 or 8
  CombineRow c;
  if (!combine_prologue(p, c)) return;
  const int lane = threadIdx.x & 31;
  float acc[CPL];
#pragma unroll
  for (int i = 0; i < CPL; ++i) acc[i] = 0.f;
  const float *src0 = p.part_o + c.prow0 * D + lane * CPL;
  for (int s0 = 0; s0 < c.ns; s0 += 4) {
    float x[4][CPL], w[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int s = s0 + u;
      const float ws = __shfl_sync(0xffffffffu, s < 32 ? c.w0 : c.w1, s & 31);
      w[u] = s < c.ns ? ws : 0.f;
      const float *src = src0 + (size_t)s * c.stride * D;
      if (s >= c.ns) {                               // (warp-uniform) past the last split: contributes exact zeros
#pragma unroll
        for (int i = 0; i < CPL; ++i) x[u][i] = 0.f;
      } else if (CPL == 2) {
        const float2 v = *reinterpret_cast<const float2 *>(src);
        x[u][0] = v.x, x[u][CPL - 1] = v.y;
      } else {
#pragma unroll
        for (int i = 0; i < CPL; i += 4) {
          const float4 v = *reinterpret_cast<const float4 *>(src + i);
          x[u][i] = v.x, x[u][(i + 1) % CPL] = v.y, x[u][(i + 2) % CPL] = v.z, x[u][(i + 3) % CPL] = v.w;
        }
      }
    }
#pragma unroll
    for (int u = 0; u < 4; ++u)
#pragma unroll
      for (int i = 0; i < CPL; ++i) acc[i] = fmaf(w[u], x[u][i], acc[i]);
  }
  uint16_t *dst = p.out + c.rowi * D + lane * CPL;
#pragma unroll
  for (int i = 0; i < CPL; i += 2) *reinterpret_cast<uint32_t *>(dst + i) = pack_bf16(acc[i] * c.inv, acc[i + 1] * c.inv);
}

// the same merge for any head_dim that is a multiple of 16 (p.head_dim; R27): a lane owns the element pairs
// 2 * lane + 64 * i of the row
__global__ void __launch_bounds__(256) attn_combine_any_kernel(const AttnParams p) {
  asm volatile("griddepcontrol.wait;" ::: "memory");
  const int d = p.head_dim;
  CombineRow c;
  if (!combine_prologue(p, c)) return;
  const int lane = threadIdx.x & 31;
  float acc[8];                                   // up to 4 pairs per lane (d <= 256)
#pragma unroll
  for (int i = 0; i < 8; ++i) acc[i] = 0.f;
  for (int s = 0; s < c.ns; ++s) {
    const float w = __shfl_sync(0xffffffffu, s < 32 ? c.w0 : c.w1, s & 31);
    const float *src = p.part_o + (c.prow0 + (size_t)s * c.stride) * d;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const int col = 2 * lane + 64 * i;
      if (col < d) {
        const float2 x = *reinterpret_cast<const float2 *>(src + col);
        acc[2 * i] = fmaf(w, x.x, acc[2 * i]);
        acc[2 * i + 1] = fmaf(w, x.y, acc[2 * i + 1]);
      }
    }
  }
  uint16_t *dst = p.out + c.rowi * d;
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int col = 2 * lane + 64 * i;
    if (col < d) *reinterpret_cast<uint32_t *>(dst + col) = pack_bf16(acc[2 * i] * c.inv, acc[2 * i + 1] * c.inv);
  }
}

template <int D, int MB>
cudaError_t launch_split_t(const AttnParams &p, cudaStream_t stream) {
  constexpr int SMEM = STAGES * 2 * BN * D * 2;
  static_assert(SMEM >= (4 * 16 * (D + 8) + 2 * 4 * 16) * 4, "merge buffer must fit in the ring");
  // the attribute is per device (fcg_config_t.device allows libraries on several GPUs in one process)
  static bool configured[64] = {};
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess) return cudaGetLastError();
  if (dev < 0 || dev >= 64 || !configured[dev]) {
    cudaError_t e = cudaFuncSetAttribute(attn_split_kernel<D, MB>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM);
    if (e != cudaSuccess) return e;
    if (dev >= 0 && dev < 64) configured[dev] = true;
  }
  dim3 grid((unsigned)(p.max_splits * p.max_row_groups), (unsigned)p.n_kv_heads, (unsigned)(p.n_layers * p.n_tasks));
  attn_split_kernel<D, MB><<<grid, NTHREADS, SMEM, stream>>>(p);
  return cudaGetLastError();
}

}  // namespace

int attn_split_ctas_per_sm(int head_dim) { return head_dim == 128 ? 2 : 4; }

cudaError_t launch_attn_split(const AttnParams &p, int head_dim, int rows_per_cta, cudaStream_t stream) {
  if (head_dim == 128) {
    if (rows_per_cta == 16) return launch_split_t<128, 1>(p, stream);
    if (rows_per_cta == 32) return launch_split_t<128, 2>(p, stream);
    if (rows_per_cta == 64) return launch_split_t<128, 4>(p, stream);
  } else if (head_dim == 64) {
    if (rows_per_cta == 16) return launch_split_t<64, 1>(p, stream);
    if (rows_per_cta == 32) return launch_split_t<64, 2>(p, stream);
    if (rows_per_cta == 64) return launch_split_t<64, 4>(p, stream);
  }
  return cudaErrorInvalidValue;
}

cudaError_t launch_attn_combine(const AttnParams &p, int head_dim, cudaStream_t stream) {
  const size_t n_rows = (size_t)p.n_layers * p.n_total * p.n_q_heads;
  const unsigned blocks = (unsigned)((n_rows + 7) / 8);
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(blocks, 1, 1);
  cfg.blockDim = dim3(256, 1, 1);
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  if (head_dim == 128) return cudaLaunchKernelEx(&cfg, attn_combine_kernel<128>, p);
  if (head_dim == 64) return cudaLaunchKernelEx(&cfg, attn_combine_kernel<64>, p);
  if (head_dim == 256) return cudaLaunchKernelEx(&cfg, attn_combine_kernel<256>, p);
  if (head_dim >= 16 && head_dim < 256 && head_dim % 16 == 0 && p.head_dim == head_dim) return cudaLaunchKernelEx(&cfg, attn_combine_any_kernel, p);
  return cudaErrorInvalidValue;
}

}  // namespace fcg
