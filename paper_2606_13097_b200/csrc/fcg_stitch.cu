// S3: fused gather + RoPE-shift (cache-stitching, Eq. 4).  The same
// kernel serves the suffix re-graft of a length-changing patch (Eq. 6, cache -> cache) and segment extraction
// (Alg. 1B `update`, cache -> segment): source and destination are strided row spaces (fcg_internal.h).
//
// HBM-bound streaming kernel: every K/V byte of a stitched segment is read once and written once.
// Work item = (chunk, layer): the tokens of one plan entry that land in one destination page, for
// one layer; the 4 warps of a CTA stride over the kv heads.  A lane owns one 16-byte column of the
// low half of a key row AND the matching 16-byte column of the high half, i.e. 8 complete rotation
// pairs (j, j + D/2) -- no shuffles.  The delta is constant per plan entry, so cos/sin depend only on
// (entry, j): 8 table entries per lane, loaded once per CTA.  No trigonometry on the device.
//
// Arithmetic (fp32 registers, error-free split of the table):
//   cos = c_hi + c_lo, sin = s_hi + s_lo with c_hi, s_hi carrying <= 16 significant bits, so the
//   products of an 8-bit bf16 input with c_hi / s_hi are EXACT in fp32.
//     x = fma(a, c_hi, -(b * s_hi))        one rounding of the exact a*c_hi - b*s_hi  (no cancellation loss)
//     x += fma(a, c_lo, -(b * s_lo))       correction, ~2^-16 of the operands
//   and likewise y = b cos + a sin.  The fp32 result is within ~2^-23 relative of the exact value;
//   RNE to bf16 then differs from the fp64 oracle by at most 1 bf16 ulp (double rounding only).
#include <cuda_bf16.h>
#include <cuda_fp16.h>

#include "fcg_internal.h"

namespace fcg {
namespace {

__device__ __forceinline__ uint4 ldg_stream(const void *p) {
  uint4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
               : "l"(p));
  return r;
}

__device__ __forceinline__ void stg_16(void *p, const uint4 &v) {
  asm volatile("st.global.L1::no_allocate.v4.u32 [%0], {%1,%2,%3,%4};" ::"l"(p), "r"(v.x), "r"(v.y), "r"(v.z),
               "r"(v.w)
               : "memory");
}

__device__ __forceinline__ float bf16_lo(uint32_t w) { return __uint_as_float(w << 16); }
__device__ __forceinline__ float bf16_hi(uint32_t w) { return __uint_as_float(w & 0xffff0000u); }

__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
  __nv_bfloat162 r = __floats2bfloat162_rn(lo, hi);  // .x = lo (low 16 bits), .y = hi
  return *reinterpret_cast<uint32_t *>(&r);
}

// rotate one pair: (a, b) -> (a cos - b sin, b cos + a sin)
__device__ __forceinline__ void rot_pair(float a, float b, const float4 &t, float &x, float &y) {
  // t = {c_hi, c_lo, s_hi, s_lo}
  const float bs = __fmul_rn(b, t.z);                 // exact
  const float as = __fmul_rn(a, t.z);                 // exact
  const float x0 = __fmaf_rn(a, t.x, -bs);            // round(a*c_hi - b*s_hi)
  const float y0 = __fmaf_rn(b, t.x, as);             // round(b*c_hi + a*s_hi)
  const float xr = __fmaf_rn(a, t.y, -__fmul_rn(b, t.w));
  const float yr = __fmaf_rn(b, t.y, __fmul_rn(a, t.w));
  x = __fadd_rn(x0, xr);
  y = __fadd_rn(y0, yr);
  // IEEE special values ("+-inf / NaN propagate"): with an infinite input the correction term is
  // inf * c_lo -- of the wrong sign, or NaN when c_lo == 0 -- and turns the infinity the definition gives into NaN.
  // A NaN result is therefore recomputed from the unsplit table (never taken for finite inputs; NaN stays NaN).
  if (__builtin_expect(x != x || y != y, 0)) {
    const float c = __fadd_rn(t.x, t.y), sn = __fadd_rn(t.z, t.w);
    x = __fmaf_rn(a, c, -__fmul_rn(b, sn));
    y = __fmaf_rn(b, c, __fmul_rn(a, sn));
  }
}

__device__ __forceinline__ void rot_word(uint32_t wa, uint32_t wb, const float4 &t0, const float4 &t1, uint32_t &oa,
                                         uint32_t &ob) {
  float x0, y0, x1, y1;
  rot_pair(bf16_lo(wa), bf16_lo(wb), t0, x0, y0);
  rot_pair(bf16_hi(wa), bf16_hi(wb), t1, x1, y1);
  oa = pack_bf16(x0, x1);
  ob = pack_bf16(y0, y1);
}

// interleaved pairs: one 32-bit word holds the pair (2j, 2j + 1)
__device__ __forceinline__ uint32_t rot_word_il(uint32_t w, const float4 &t) {
  float x, y;
  rot_pair(bf16_lo(w), bf16_hi(w), t, x, y);
  return pack_bf16(x, y);
}

// ---- fp8 (e4m3) source rows, R26 ---------------------------------------------------------
__device__ __forceinline__ uint2 ldg_stream8(const void *p) {
  uint2 r;
  asm volatile("ld.global.nc.L1::no_allocate.v2.u32 {%0,%1}, [%2];" : "=r"(r.x), "=r"(r.y) : "l"(p));
  return r;
}
// two e4m3 codes -> two floats (exact: e4m3 is a subset of fp16)
__device__ __forceinline__ float2 e4m3x2_to_float2(uint32_t two_codes) {
  uint32_t h2;
  asm("{cvt.rn.f16x2.e4m3x2 %0, %1;}" : "=r"(h2) : "h"((unsigned short)two_codes));
  return __half22float2(*reinterpret_cast<__half2 *>(&h2));
}
// 2^(eb - 127) for a scale byte eb in [0, 254] (0 -> the subnormal 2^-127)
__device__ __forceinline__ float scale_of(uint32_t eb) { return __uint_as_float(eb ? (eb << 23) : 0x00400000u); }
// 8 codes (two 32-bit words) -> 8 de-quantised floats: value(code) * 2^e, exact in fp32
__device__ __forceinline__ void dequant8(const uint2 &c, float sc, float *out) {
  const float2 a = e4m3x2_to_float2(c.x & 0xffffu), b = e4m3x2_to_float2(c.x >> 16);
  const float2 d = e4m3x2_to_float2(c.y & 0xffffu), e = e4m3x2_to_float2(c.y >> 16);
  out[0] = a.x * sc, out[1] = a.y * sc, out[2] = b.x * sc, out[3] = b.y * sc;
  out[4] = d.x * sc, out[5] = d.y * sc, out[6] = e.x * sc, out[7] = e.y * sc;
}
__device__ __forceinline__ uint4 pack8(const float *x) {
  return make_uint4(pack_bf16(x[0], x[1]), pack_bf16(x[2], x[3]), pack_bf16(x[4], x[5]), pack_bf16(x[6], x[7]));
}

// The body of one entry whose source is an fp8 segment: same work split as the bf16 path (a lane owns the 8 low-half and
// the 8 matching high-half elements of a row), rows are D code bytes + one scale byte.  K: de-quantise, rotate with the
// compensated fp32 scheme (a de-quantised element has <= 4 significant bits, so its products with c_hi / s_hi are exact
// as for bf16 inputs), ONE rounding to bf16.  V: de-quantise, round to bf16 (exact outside the deepest subnormals).
// DT = 0: head_dim at run time (`Dr`, any multiple of 16 up to 256; lanes beyond TPS * LPT idle)
template <int DT>
__device__ __forceinline__ void stitch_fp8_rows(const StitchEntryDev &en, const StitchChunkDev &ch, int layer, int Hkv, int warp,
                                                int col, int tl, bool rotate, bool il, const float4 *tab, int Dr) {
  const int D = DT ? DT : Dr;
  const int LPT = D / 16, TPS = 32 / LPT;
  constexpr int STEPS = 4, HEADS = 2;
  const int ntok = DT ? ch.ntok : (tl < TPS ? ch.ntok : 0);   // an idle lane sees an empty chunk
  // a code row is half a bf16 row: two kv heads per pass keep as many bytes in flight per lane as the bf16 path has
  for (int g0 = warp; g0 < Hkv; g0 += 4 * HEADS) {
    for (int t0 = 0; t0 < ntok; t0 += TPS * STEPS) {
      uint2 klo[HEADS][STEPS], khi[HEADS][STEPS], vlo[HEADS][STEPS], vhi[HEADS][STEPS];
      uint32_t ke[HEADS][STEPS], ve[HEADS][STEPS];
#pragma unroll
      for (int h = 0; h < HEADS; ++h) {
        const int g = g0 + 4 * h;
        if (g < Hkv) {
          const size_t src_row = (size_t)layer * (size_t)en.src_layer_stride + (size_t)g * (size_t)en.src_head_stride + (size_t)ch.src_tok;
          const char *ksrc = reinterpret_cast<const char *>(en.k_src) + src_row * D + col * 8;
          const char *vsrc = reinterpret_cast<const char *>(en.v_src) + src_row * D + col * 8;
          const uint8_t *kexp = reinterpret_cast<const uint8_t *>(en.k_exp) + src_row;
          const uint8_t *vexp = reinterpret_cast<const uint8_t *>(en.v_exp) + src_row;
#pragma unroll
          for (int s = 0; s < STEPS; ++s) {
            const int t = t0 + s * TPS + tl;
            if (t < ntok) {
              const size_t off = (size_t)t * D;
              klo[h][s] = ldg_stream8(ksrc + off);
              khi[h][s] = ldg_stream8(ksrc + off + D / 2);
              vlo[h][s] = ldg_stream8(vsrc + off);
              vhi[h][s] = ldg_stream8(vsrc + off + D / 2);
              ke[h][s] = __ldg(kexp + t);
              ve[h][s] = __ldg(vexp + t);
            }
          }
        }
      }
#pragma unroll
      for (int h = 0; h < HEADS; ++h) {
        const int g = g0 + 4 * h;
        if (g < Hkv) {
          const size_t dst_row = (size_t)layer * (size_t)en.dst_layer_stride + (size_t)g * (size_t)en.dst_head_stride + (size_t)ch.dst_tok;
          char *kdst = reinterpret_cast<char *>(en.k_dst) + dst_row * (D * 2) + col * 16;
          char *vdst = reinterpret_cast<char *>(en.v_dst) + dst_row * (D * 2) + col * 16;
#pragma unroll
          for (int s = 0; s < STEPS; ++s) {
            const int t = t0 + s * TPS + tl;
            if (t < ntok) {
              const size_t off = (size_t)t * (D * 2);
              float a[8], b[8];
              dequant8(klo[h][s], scale_of(ke[h][s]), a);
              dequant8(khi[h][s], scale_of(ke[h][s]), b);
              if (rotate) {
                float x[8], y[8];
                if (!il) {
#pragma unroll
                  for (int i = 0; i < 8; ++i) rot_pair(a[i], b[i], tab[i], x[i], y[i]);
                } else {
#pragma unroll
                  for (int i = 0; i < 4; ++i) {
                    rot_pair(a[2 * i], a[2 * i + 1], tab[i], x[2 * i], x[2 * i + 1]);
                    rot_pair(b[2 * i], b[2 * i + 1], tab[4 + i], y[2 * i], y[2 * i + 1]);
                  }
                }
                stg_16(kdst + off, pack8(x));
                stg_16(kdst + off + D, pack8(y));
              } else {
                stg_16(kdst + off, pack8(a));
                stg_16(kdst + off + D, pack8(b));
              }
              dequant8(vlo[h][s], scale_of(ve[h][s]), a);
              dequant8(vhi[h][s], scale_of(ve[h][s]), b);
              stg_16(vdst + off, pack8(a));
              stg_16(vdst + off + D, pack8(b));
            }
          }
        }
      }
    }
  }
}

template <int DT, bool FP8>
__global__ void __launch_bounds__(128, FP8 ? 3 : 4) stitch_kernel(const StitchParams p) {
  // DT = 0: head_dim at run time (p.head_dim: any multiple of 16 up to 256, R27); the lanes beyond TPS * LPT idle
  const int D = DT ? DT : p.head_dim;
  const int LPT = D / 16;          // lanes per token: one 16-byte column of each half per lane
  const int TPS = 32 / LPT;        // tokens per warp step
  constexpr int STEPS = 4;         // steps in flight per batch (4 x 64 B per lane)
  const int ROW_BYTES = D * 2;

  const StitchChunkDev ch = p.chunks[blockIdx.x];
  const StitchEntryDev en = p.entries[ch.entry];
  const int layer = blockIdx.y;
  const int lane = threadIdx.x & 31;
  const int warp = threadIdx.x >> 5;
  const int col = lane % LPT;
  const int tl = lane / LPT;
  const int ntok = DT ? ch.ntok : (tl < TPS ? ch.ntok : 0);   // an idle lane sees an empty chunk
  const bool rotate = en.table_off >= 0;
  const bool il = p.interleaved != 0;

  // the lane's two 16-byte vectors of a key row: elements [col*8, col*8+8) and [D/2 + col*8, D/2 + col*8 + 8).
  // half-split: pair i of the lane = (lo[i], hi[i]) with frequency col*8 + i;
  // interleaved: pairs (lo[2i], lo[2i+1]) with frequency col*4 + i and (hi[2i], hi[2i+1]) with D/4 + col*4 + i.
  float4 tab[8];
  if (rotate) {
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const int j = il ? ((i >> 2) * (D / 4) + col * 4 + (i & 3)) : (col * 8 + i);
      tab[i] = __ldg(p.table + en.table_off + j);
    }
  }

  const int Hkv = p.n_kv_heads;
  if (FP8 && en.src_fp8) {           // (the bf16 instantiation carries no fp8 code: its registers and SASS stay as they were)
    stitch_fp8_rows<DT>(en, ch, layer, Hkv, warp, col, tl, rotate, il, tab, D);
    return;
  }
  for (int g = warp; g < Hkv; g += 4) {
    const size_t src_row = (size_t)layer * (size_t)en.src_layer_stride + (size_t)g * (size_t)en.src_head_stride + (size_t)ch.src_tok;
    const size_t dst_row = (size_t)layer * (size_t)en.dst_layer_stride + (size_t)g * (size_t)en.dst_head_stride + (size_t)ch.dst_tok;
    const char *ksrc = reinterpret_cast<const char *>(en.k_src) + src_row * ROW_BYTES + col * 16;
    const char *vsrc = reinterpret_cast<const char *>(en.v_src) + src_row * ROW_BYTES + col * 16;
    char *kdst = reinterpret_cast<char *>(en.k_dst) + dst_row * ROW_BYTES + col * 16;
    char *vdst = reinterpret_cast<char *>(en.v_dst) + dst_row * ROW_BYTES + col * 16;

    for (int t0 = 0; t0 < ntok; t0 += TPS * STEPS) {
      uint4 klo[STEPS], khi[STEPS], vlo[STEPS], vhi[STEPS];
#pragma unroll
      for (int s = 0; s < STEPS; ++s) {
        const int t = t0 + s * TPS + tl;
        if (t < ntok) {
          const size_t off = (size_t)t * ROW_BYTES;
          klo[s] = ldg_stream(ksrc + off);
          khi[s] = ldg_stream(ksrc + off + D);
          vlo[s] = ldg_stream(vsrc + off);
          vhi[s] = ldg_stream(vsrc + off + D);
        }
      }
#pragma unroll
      for (int s = 0; s < STEPS; ++s) {
        const int t = t0 + s * TPS + tl;
        if (t < ntok) {
          const size_t off = (size_t)t * ROW_BYTES;
          uint4 olo = klo[s], ohi = khi[s];
          if (rotate) {
            if (!il) {
              rot_word(klo[s].x, khi[s].x, tab[0], tab[1], olo.x, ohi.x);
              rot_word(klo[s].y, khi[s].y, tab[2], tab[3], olo.y, ohi.y);
              rot_word(klo[s].z, khi[s].z, tab[4], tab[5], olo.z, ohi.z);
              rot_word(klo[s].w, khi[s].w, tab[6], tab[7], olo.w, ohi.w);
            } else {
              olo.x = rot_word_il(klo[s].x, tab[0]);
              olo.y = rot_word_il(klo[s].y, tab[1]);
              olo.z = rot_word_il(klo[s].z, tab[2]);
              olo.w = rot_word_il(klo[s].w, tab[3]);
              ohi.x = rot_word_il(khi[s].x, tab[4]);
              ohi.y = rot_word_il(khi[s].y, tab[5]);
              ohi.z = rot_word_il(khi[s].z, tab[6]);
              ohi.w = rot_word_il(khi[s].w, tab[7]);
            }
          }
          stg_16(kdst + off, olo);
          stg_16(kdst + off + D, ohi);
          stg_16(vdst + off, vlo[s]);
          stg_16(vdst + off + D, vhi[s]);
        }
      }
    }
  }
}

// q / k rows of the patch tokens -> rotated to their absolute positions (fcg_patch_rope).  One CTA per (token, layer);
// a thread owns the two 16-byte vectors [col*8, +8) and [D/2 + col*8, +8) of one head row, as in stitch_kernel.
template <int DT>
__global__ void __launch_bounds__(128) rope_qk_kernel(const RopeQkParams p) {
  const int D = DT ? DT : p.head_dim;      // DT = 0: head_dim at run time
  const int LPT = D / 16;
  const int tok = blockIdx.x, layer = blockIdx.y;
  const int rows = p.n_q_heads + p.n_kv_heads;
  const bool il = p.interleaved != 0;
  for (int w = threadIdx.x; w < rows * LPT; w += blockDim.x) {
    const int r = w / LPT, col = w % LPT;
    const bool is_q = r < p.n_q_heads;
    const size_t row = is_q ? ((size_t)layer * p.n_total + tok) * p.n_q_heads + r
                            : ((size_t)layer * p.n_total + tok) * p.n_kv_heads + (r - p.n_q_heads);
    const char *src = reinterpret_cast<const char *>(is_q ? p.q : p.k) + row * (D * 2) + col * 16;
    char *dst = reinterpret_cast<char *>(is_q ? p.q_out : p.k_out) + row * (D * 2) + col * 16;
    const uint4 lo = *reinterpret_cast<const uint4 *>(src), hi = *reinterpret_cast<const uint4 *>(src + D);
    float4 tab[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const int j = il ? ((i >> 2) * (D / 4) + col * 4 + (i & 3)) : (col * 8 + i);
      tab[i] = __ldg(p.table + (size_t)tok * (D / 2) + j);
    }
    uint4 olo, ohi;
    if (!il) {
      rot_word(lo.x, hi.x, tab[0], tab[1], olo.x, ohi.x);
      rot_word(lo.y, hi.y, tab[2], tab[3], olo.y, ohi.y);
      rot_word(lo.z, hi.z, tab[4], tab[5], olo.z, ohi.z);
      rot_word(lo.w, hi.w, tab[6], tab[7], olo.w, ohi.w);
    } else {
      olo.x = rot_word_il(lo.x, tab[0]);
      olo.y = rot_word_il(lo.y, tab[1]);
      olo.z = rot_word_il(lo.z, tab[2]);
      olo.w = rot_word_il(lo.w, tab[3]);
      ohi.x = rot_word_il(hi.x, tab[4]);
      ohi.y = rot_word_il(hi.y, tab[5]);
      ohi.z = rot_word_il(hi.z, tab[6]);
      ohi.w = rot_word_il(hi.w, tab[7]);
    }
    *reinterpret_cast<uint4 *>(dst) = olo;
    *reinterpret_cast<uint4 *>(dst + D) = ohi;
  }
}

}  // namespace

cudaError_t launch_rope_qk(const RopeQkParams &p, int head_dim, cudaStream_t stream) {
  if (p.n_total <= 0 || p.n_layers <= 0) return cudaSuccess;
  dim3 grid((unsigned)p.n_total, (unsigned)p.n_layers, 1);
  if (head_dim == 128)
    rope_qk_kernel<128><<<grid, 128, 0, stream>>>(p);
  else if (head_dim == 64)
    rope_qk_kernel<64><<<grid, 128, 0, stream>>>(p);
  else if (head_dim == 256)
    rope_qk_kernel<256><<<grid, 128, 0, stream>>>(p);
  else if (head_dim >= 16 && head_dim < 256 && head_dim % 16 == 0 && p.head_dim == head_dim)
    rope_qk_kernel<0><<<grid, 128, 0, stream>>>(p);
  else
    return cudaErrorInvalidValue;
  return cudaGetLastError();
}

cudaError_t launch_stitch(const StitchParams &p, int head_dim, cudaStream_t stream) {
  if (p.n_chunks <= 0) return cudaSuccess;
  dim3 grid((unsigned)p.n_chunks, (unsigned)p.n_layers, 1);
  dim3 block(128, 1, 1);
  if (head_dim == 128) {
    if (p.any_fp8)
      stitch_kernel<128, true><<<grid, block, 0, stream>>>(p);
    else
      stitch_kernel<128, false><<<grid, block, 0, stream>>>(p);
  } else if (head_dim == 64) {
    if (p.any_fp8)
      stitch_kernel<64, true><<<grid, block, 0, stream>>>(p);
    else
      stitch_kernel<64, false><<<grid, block, 0, stream>>>(p);
  } else if (head_dim == 256) {
    if (p.any_fp8)
      stitch_kernel<256, true><<<grid, block, 0, stream>>>(p);
    else
      stitch_kernel<256, false><<<grid, block, 0, stream>>>(p);
  } else if (head_dim >= 16 && head_dim < 256 && head_dim % 16 == 0 && p.head_dim == head_dim) {
    if (p.any_fp8)
      stitch_kernel<0, true><<<grid, block, 0, stream>>>(p);
    else
      stitch_kernel<0, false><<<grid, block, 0, stream>>>(p);
  } else {
    return cudaErrorInvalidValue;
  }
  return cudaGetLastError();
}

}  // namespace fcg
