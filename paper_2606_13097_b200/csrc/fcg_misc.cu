// Small bit-copy kernels: S1 segment registration (strided source -> contiguous library slot),
// S4 patch K/V scatter (Eq. 6: the recomputed span is written into the cache),
// and the dense read-back of a task's cache through its page table.  All are 16-byte vectorised
// row copies; none does arithmetic on the payload.
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
