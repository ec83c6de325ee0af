// Small bit-copy kernels: S1 segment registration (strided source -> contiguous library slot),
// S4 patch K/V scatter (Eq. 6: the recomputed span is written into the cache),
// and the dense read-back of a task's cache through its page table.  All are 16-byte vectorised
// row copies; none does arithmetic on the payload.
#include <cuda_fp8.h>

#include "fcg_internal.h"

namespace fcg {
namespace {

__device__ __forceinline__ uint4 ld16(const void *p) { return *reinterpret_cast<const uint4 *>(p); }
__device__ __forceinline__ void st16(void *p, const uint4 &v) { *reinterpret_cast<uint4 *>(p) = v; }

// one row = head_dim bf16 = head_dim/8 16-byte vectors; a thread copies one vector of K and of V
__global__ void __launch_bounds__(256) register_copy_kernel(const RegisterParams p) {
  const int vpr = p.head_dim >> 3;
  const size_t total = (size_t)p.n_layers * p.n_kv_heads * p.n_tokens * vpr;
  for (size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (size_t)gridDim.x * blockDim.x) {
    const int vec = (int)(idx % vpr);
    size_t row = idx / vpr;
    const int t = (int)(row % p.n_tokens);
    row /= p.n_tokens;
    const int h = (int)(row % p.n_kv_heads);
    const int l = (int)(row / p.n_kv_heads);
    const size_t src = (size_t)((int64_t)l * p.s_layer + (int64_t)h * p.s_head + (int64_t)t * p.s_tok) + (size_t)vec * 8;
    const size_t dst = idx * 8;
    st16(p.k_dst + dst, ld16(p.k_src + src));
    st16(p.v_dst + dst, ld16(p.v_src + src));
  }
}

// S1, fp8 storage (R26): one warp per row of D bf16 elements.  e = the smallest integer with amax <= 448 * 2^e
// (amax over the finite elements; integer arithmetic on the exponent field: 448 = 1.75 * 2^8), clamped to [-127, 127],
// 0 for an all-zero row; code = RNE_e4m3(x * 2^-e) (the scaling is exact), non-finite elements -> the NaN code 0x7F.
template <int D>
__global__ void __launch_bounds__(256) register_fp8_kernel(const RegisterFp8Params p) {
  constexpr int EPL = D / 32;                         // elements per lane: 8 (D = 256), 4 (D = 128) or 2 (D = 64)
  const size_t n_rows = (size_t)p.n_layers * p.n_kv_heads * p.n_tokens;
  const int lane = threadIdx.x & 31;
  for (size_t row = (size_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); row < 2 * n_rows;
       row += (size_t)gridDim.x * (blockDim.x >> 5)) {
    const bool is_v = row >= n_rows;
    const size_t r = is_v ? row - n_rows : row;
    const int t = (int)(r % p.n_tokens);
    const size_t lh = r / p.n_tokens;
    const int h = (int)(lh % p.n_kv_heads), l = (int)(lh / p.n_kv_heads);
    const uint16_t *src = (is_v ? p.v_src : p.k_src) + (size_t)((int64_t)l * p.s_layer + (int64_t)h * p.s_head + (int64_t)t * p.s_tok) + lane * EPL;
    float x[EPL];
    {
      uint32_t w[EPL / 2];
      if (EPL == 8) {
        const uint4 v = *reinterpret_cast<const uint4 *>(src);
        w[0] = v.x, w[EPL / 2 > 1 ? 1 : 0] = v.y, w[EPL / 2 > 2 ? 2 : 0] = v.z, w[EPL / 2 > 3 ? 3 : 0] = v.w;
      } else if (EPL == 4) {
        const uint2 v = *reinterpret_cast<const uint2 *>(src);
        w[0] = v.x, w[EPL / 2 > 1 ? 1 : 0] = v.y;
      } else {
        w[0] = *reinterpret_cast<const uint32_t *>(src);
      }
#pragma unroll
      for (int i = 0; i < EPL / 2; ++i) x[2 * i] = __uint_as_float(w[i] << 16), x[2 * i + 1] = __uint_as_float(w[i] & 0xffff0000u);
    }
    uint32_t amax = 0;                                // |x| as bits: ordered like the values for non-negative floats
#pragma unroll
    for (int i = 0; i < EPL; ++i) {
      const uint32_t a = __float_as_uint(x[i]) & 0x7fffffffu;
      if (a < 0x7f800000u) amax = max(amax, a);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) amax = max(amax, __shfl_xor_sync(0xffffffffu, amax, o));
    int e = 0;
    if (amax != 0) {
      const int be = (int)(amax >> 23);               // biased exponent; 0 = subnormal: far below 448 * 2^-127 -> clamps
      e = be == 0 ? -127 : (be - 127) - ((amax & 0x7fffffu) <= 0x600000u ? 8 : 7);
      e = max(-127, min(127, e));
    }
    uint64_t packed = 0;
#pragma unroll
    for (int i = 0; i < EPL; i += 2) {
      const float a = scalbnf(x[i], -e), b = scalbnf(x[i + 1], -e);
      uint32_t c2 = (uint32_t)__nv_cvt_float2_to_fp8x2(make_float2(a, b), __NV_SATFINITE, __NV_E4M3);
      if ((__float_as_uint(x[i]) & 0x7fffffffu) >= 0x7f800000u) c2 = (c2 & 0xff00u) | 0x7fu;
      if ((__float_as_uint(x[i + 1]) & 0x7fffffffu) >= 0x7f800000u) c2 = (c2 & 0x00ffu) | 0x7f00u;
      packed |= (uint64_t)c2 << (8 * i);
    }
    uint8_t *dst = (is_v ? p.v_dst : p.k_dst) + r * D + lane * EPL;
    if (EPL == 8)
      *reinterpret_cast<uint2 *>(dst) = make_uint2((uint32_t)packed, (uint32_t)(packed >> 32));
    else if (EPL == 4)
      *reinterpret_cast<uint32_t *>(dst) = (uint32_t)packed;
    else
      *reinterpret_cast<uint16_t *>(dst) = (uint16_t)packed;
    if (lane == 0) (is_v ? p.v_exp : p.k_exp)[r] = (uint8_t)(e + 127);
  }
}

// the same for any head_dim that is a multiple of 8 (p.head_dim <= 256): lane c owns the elements [8c, 8c + 8) of the row
__global__ void __launch_bounds__(256) register_fp8_any_kernel(const RegisterFp8Params p) {
  const int D = p.head_dim;
  const size_t n_rows = (size_t)p.n_layers * p.n_kv_heads * p.n_tokens;
  const int lane = threadIdx.x & 31;
  const bool on = lane * 8 < D;
  for (size_t row = (size_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); row < 2 * n_rows;
       row += (size_t)gridDim.x * (blockDim.x >> 5)) {
    const bool is_v = row >= n_rows;
    const size_t r = is_v ? row - n_rows : row;
    const int t = (int)(r % p.n_tokens);
    const size_t lh = r / p.n_tokens;
    const int h = (int)(lh % p.n_kv_heads), l = (int)(lh / p.n_kv_heads);
    const uint16_t *src = (is_v ? p.v_src : p.k_src) + (size_t)((int64_t)l * p.s_layer + (int64_t)h * p.s_head + (int64_t)t * p.s_tok) + lane * 8;
    float x[8];
    uint32_t amax = 0;
    if (on) {
      const uint4 v = *reinterpret_cast<const uint4 *>(src);
      const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
      for (int i = 0; i < 4; ++i) x[2 * i] = __uint_as_float(w[i] << 16), x[2 * i + 1] = __uint_as_float(w[i] & 0xffff0000u);
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        const uint32_t a = __float_as_uint(x[i]) & 0x7fffffffu;
        if (a < 0x7f800000u) amax = max(amax, a);
      }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) amax = max(amax, __shfl_xor_sync(0xffffffffu, amax, o));
    int e = 0;
    if (amax != 0) {
      const int be = (int)(amax >> 23);
      e = be == 0 ? -127 : (be - 127) - ((amax & 0x7fffffu) <= 0x600000u ? 8 : 7);
      e = max(-127, min(127, e));
    }
    if (on) {
      uint64_t packed = 0;
#pragma unroll
      for (int i = 0; i < 8; i += 2) {
        const float a = scalbnf(x[i], -e), b = scalbnf(x[i + 1], -e);
        uint32_t c2 = (uint32_t)__nv_cvt_float2_to_fp8x2(make_float2(a, b), __NV_SATFINITE, __NV_E4M3);
        if ((__float_as_uint(x[i]) & 0x7fffffffu) >= 0x7f800000u) c2 = (c2 & 0xff00u) | 0x7fu;
        if ((__float_as_uint(x[i + 1]) & 0x7fffffffu) >= 0x7f800000u) c2 = (c2 & 0x00ffu) | 0x7f00u;
        packed |= (uint64_t)c2 << (8 * i);
      }
      uint8_t *dst = (is_v ? p.v_dst : p.k_dst) + r * D + lane * 8;
      *reinterpret_cast<uint2 *>(dst) = make_uint2((uint32_t)packed, (uint32_t)(packed >> 32));
    }
    if (lane == 0) (is_v ? p.v_exp : p.k_exp)[r] = (uint8_t)(e + 127);
  }
}

__global__ void __launch_bounds__(256) scatter_kernel(const ScatterParams p) {
  // the attention kernel that follows may start its prologue now (it waits for this grid before reading the cache)
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  const int vpr = p.head_dim >> 3;
  const size_t total = (size_t)p.n_layers * p.n_total * p.n_kv_heads * vpr;
  for (size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (size_t)gridDim.x * blockDim.x) {
    const int vec = (int)(idx % vpr);
    size_t row = idx / vpr;
    const int g = (int)(row % p.n_kv_heads);
    row /= p.n_kv_heads;
    const int i = (int)(row % p.n_total);
    const int li = (int)(row / p.n_total);
    const int pos = p.positions[i];
    const int page = p.tables[p.tok_table_off[i] + pos / p.page_size];
    const int slot = pos % p.page_size;
    const size_t dst =
        ((((size_t)(p.layer_begin + li) * p.n_pages + (size_t)page) * p.n_kv_heads + g) * p.page_size + slot) *
            (size_t)p.head_dim + (size_t)vec * 8;
    st16(p.k_pool + dst, ld16(p.k_new + idx * 8));
    st16(p.v_pool + dst, ld16(p.v_new + idx * 8));
  }
}

__global__ void __launch_bounds__(256) task_read_kernel(const ReadParams p) {
  const int vpr = p.head_dim >> 3;
  const size_t total = (size_t)p.n_kv_heads * p.n * vpr;
  for (size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (size_t)gridDim.x * blockDim.x) {
    const int vec = (int)(idx % vpr);
    size_t row = idx / vpr;
    const int t = (int)(row % p.n);
    const int g = (int)(row / p.n);
    const int pos = p.begin + t;
    const int page = p.table[pos / p.page_size];
    const int slot = pos % p.page_size;
    const size_t src = ((((size_t)p.layer * p.n_pages + (size_t)page) * p.n_kv_heads + g) * p.page_size + slot) *
                           (size_t)p.head_dim + (size_t)vec * 8;
    st16(p.k_out + idx * 8, ld16(p.k_pool + src));
    st16(p.v_out + idx * 8, ld16(p.v_pool + src));
  }
}

inline unsigned grid_for(size_t total_threads) {
  size_t blocks = (total_threads + 255) / 256;
  const size_t cap = 148u * 16u;
  if (blocks > cap) blocks = cap;
  if (blocks == 0) blocks = 1;
  return (unsigned)blocks;
}

}  // namespace

cudaError_t launch_register_copy(const RegisterParams &p, cudaStream_t stream) {
  const size_t total = (size_t)p.n_layers * p.n_kv_heads * p.n_tokens * (p.head_dim >> 3);
  register_copy_kernel<<<grid_for(total), 256, 0, stream>>>(p);
  return cudaGetLastError();
}

cudaError_t launch_register_fp8(const RegisterFp8Params &p, cudaStream_t stream) {
  const size_t rows = 2 * (size_t)p.n_layers * p.n_kv_heads * p.n_tokens;
  const unsigned grid = grid_for(rows * 32);
  if (p.head_dim == 128)
    register_fp8_kernel<128><<<grid, 256, 0, stream>>>(p);
  else if (p.head_dim == 64)
    register_fp8_kernel<64><<<grid, 256, 0, stream>>>(p);
  else if (p.head_dim == 256)
    register_fp8_kernel<256><<<grid, 256, 0, stream>>>(p);
  else if (p.head_dim >= 8 && p.head_dim < 256 && p.head_dim % 8 == 0)
    register_fp8_any_kernel<<<grid, 256, 0, stream>>>(p);
  else
    return cudaErrorInvalidValue;
  return cudaGetLastError();
}

cudaError_t launch_scatter(const ScatterParams &p, cudaStream_t stream) {
  const size_t total = (size_t)p.n_layers * p.n_total * p.n_kv_heads * (p.head_dim >> 3);
  scatter_kernel<<<grid_for(total), 256, 0, stream>>>(p);
  return cudaGetLastError();
}

cudaError_t launch_task_read(const ReadParams &p, cudaStream_t stream) {
  const size_t total = (size_t)p.n_kv_heads * p.n * (p.head_dim >> 3);
  task_read_kernel<<<grid_for(total), 256, 0, stream>>>(p);
  return cudaGetLastError();
}

}  // namespace fcg
