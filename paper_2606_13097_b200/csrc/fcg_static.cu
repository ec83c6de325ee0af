// fcg_segment_shift_static: the gather + RoPE-shift kernel (S3, Eq. 4) for callers that must not
// allocate device memory.  Contract and rationale: include/fcg.h.
//
// The library path (fcg_stitch) keeps the kernel's device-side plan -- one entry descriptor, the chunk list and the
// cos/sin table of the delta -- in the workspace of an arena somebody had to allocate.  Here the same plan lives in a
// file-scope device array that comes with the loaded library image, so the call itself needs no allocation at all:
//
//   static_plan_kernel   writes the plan of THIS call into g_static_plan (device code names the array directly);
//                        entry and table arrive as kernel parameters, the chunk list is generated on the device
//   stitch_kernel        the unchanged product kernel (fcg_stitch.cu, launch_stitch), pointed at the array through
//                        the device address that cudaGetSymbolAddress returned
//
// In host code `g_static_plan` is only a handle for the runtime: it is never dereferenced or handed to a kernel here.
// The device address is looked up once per device (with that device current) and cached.
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <stdint.h>
#include <string.h>

#include <mutex>

#include "../../include/fcg.h"
#include "fcg_internal.h"

namespace {

constexpr int MAX_TOKENS = 65536;                 // FCG_STATIC_SHIFT_MAX_TOKENS of fcg.h
constexpr int CHUNK_TOKENS = 16;                  // tokens per work item, as one page of the library path
constexpr int MAX_CHUNKS = MAX_TOKENS / CHUNK_TOKENS;
constexpr int MAX_HALF = 128;                     // head_dim <= 256
constexpr size_t OFF_ENTRY = 0;                                                  // one StitchEntryDev (80 B)
constexpr size_t OFF_TABLE = 256;                                                // MAX_HALF float4
constexpr size_t OFF_CHUNKS = OFF_TABLE + MAX_HALF * sizeof(float4);             // MAX_CHUNKS StitchChunkDev
constexpr size_t PLAN_BYTES = OFF_CHUNKS + MAX_CHUNKS * sizeof(fcg::StitchChunkDev);   // 67 840 B per device
static_assert(sizeof(fcg::StitchEntryDev) <= OFF_TABLE && OFF_CHUNKS % 256 == 0, "plan layout");
static_assert(FCG_STATIC_SHIFT_MAX_TOKENS == MAX_TOKENS, "fcg.h states the limit");

// The scratch of this entry point.  Every device that loads libfcg.so carries these 66 KB until the process exits.
static __device__ __align__(256) unsigned char g_static_plan[PLAN_BYTES];

struct PlanArgs {                                 // 2 144 B of kernel parameters (limit 4 KB)
  fcg::StitchEntryDev entry;
  float4 table[MAX_HALF];
  int32_t n_tokens, n_table;
};

// Rewrites every byte of the plan that the following stitch_kernel launch reads: nothing of the previous call's plan
// is relied upon, and nothing has to start at zero.
__global__ void __launch_bounds__(256) static_plan_kernel(const __grid_constant__ PlanArgs a) {
  fcg::StitchEntryDev *entry = reinterpret_cast<fcg::StitchEntryDev *>(g_static_plan + OFF_ENTRY);
  float4 *table = reinterpret_cast<float4 *>(g_static_plan + OFF_TABLE);
  fcg::StitchChunkDev *chunks = reinterpret_cast<fcg::StitchChunkDev *>(g_static_plan + OFF_CHUNKS);
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i == 0) *entry = a.entry;
  if (i < a.n_table) table[i] = a.table[i];
  const int n_chunks = (a.n_tokens + CHUNK_TOKENS - 1) / CHUNK_TOKENS;
  if (i < n_chunks) {
    fcg::StitchChunkDev c;
    c.entry = 0;
    c.dst_tok = c.src_tok = i * CHUNK_TOKENS;     // source and destination are both dense [L][Hkv][n][D]
    c.ntok = min(CHUNK_TOKENS, a.n_tokens - i * CHUNK_TOKENS);
    chunks[i] = c;
  }
}

constexpr int MAX_DEVICES = 64;
std::mutex g_mu;
unsigned char *g_plan_dev[MAX_DEVICES];           // device address of g_static_plan per device ordinal (NULL: not set up)

fcg_status_t fail(fcg_status_t st, const char *fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  fcg::set_last_error(buf);
  return st;
}

// same hi / lo split as the library path's table (fcg_api.cu GatherBuilder::table_for): hi carries 16 significant
// bits so that bf16 x hi is exact in fp32
void split(double x, float &hi, float &lo) {
  float f = (float)x;
  uint32_t b;
  memcpy(&b, &f, 4);
  b = (b + 0x80u) & 0xffffff00u;
  memcpy(&hi, &b, 4);
  lo = (float)(x - (double)hi);
}

bool overlap(const void *a, const void *b, uint64_t bytes) {
  const uintptr_t x = (uintptr_t)a, y = (uintptr_t)b;
  return x < y + bytes && y < x + bytes;
}

}  // namespace

extern "C" {

int32_t fcg_segment_shift_static_max_tokens(void) { return MAX_TOKENS; }

fcg_status_t fcg_segment_shift_static(const void *k_src, const void *v_src, void *k_dst, void *v_dst, int32_t n_layers,
                                      int32_t n_kv_heads, int32_t n_tokens, int32_t head_dim, int32_t rope_mode,
                                      double rope_base, const double *inv_freq, int32_t delta, void *stream) {
  // ---- host-side checks: all of them before anything is enqueued ----
  if (n_layers <= 0 || n_layers > 65535 || n_kv_heads <= 0 || n_tokens < 0)
    return fail(FCG_ERR_INVALID_ARG, "fcg_segment_shift_static: bad shape (n_layers %d in [1, 65535], n_kv_heads %d > 0, n_tokens %d >= 0)",
                n_layers, n_kv_heads, n_tokens);
  if (head_dim < 16 || head_dim > 256 || head_dim % 16)
    return fail(FCG_ERR_INVALID_ARG, "fcg_segment_shift_static: head_dim %d is not a multiple of 16 in [16, 256]", head_dim);
  if (rope_mode != FCG_ROPE_NONE && rope_mode != FCG_ROPE_HALF_SPLIT && rope_mode != FCG_ROPE_INTERLEAVED)
    return fail(FCG_ERR_INVALID_ARG, "fcg_segment_shift_static: unknown rope_mode %d", rope_mode);
  if (rope_mode != FCG_ROPE_NONE && !inv_freq && !(rope_base > 0.0))
    return fail(FCG_ERR_INVALID_ARG, "fcg_segment_shift_static: rope_base must be > 0 when inv_freq is NULL");
  if (n_tokens > MAX_TOKENS)
    return fail(FCG_ERR_RANGE, "fcg_segment_shift_static: %d tokens exceed the static plan's limit of %d per call "
                "(split the segment, or use fcg_stitch)", n_tokens, MAX_TOKENS);
  if (n_tokens == 0) return FCG_OK;
  if (!k_src || !v_src || !k_dst || !v_dst) return fail(FCG_ERR_INVALID_ARG, "fcg_segment_shift_static: NULL buffer");
  if (((uintptr_t)k_src | (uintptr_t)v_src | (uintptr_t)k_dst | (uintptr_t)v_dst) & 15)
    return fail(FCG_ERR_INVALID_ARG, "fcg_segment_shift_static: buffers must be 16-byte aligned");
  const uint64_t bytes = (uint64_t)n_layers * n_kv_heads * (uint64_t)n_tokens * head_dim * 2;
  if (overlap(k_src, k_dst, bytes) || overlap(k_src, v_dst, bytes) || overlap(v_src, k_dst, bytes) ||
      overlap(v_src, v_dst, bytes) || overlap(k_dst, v_dst, bytes))
    return fail(FCG_ERR_OVERLAP, "fcg_segment_shift_static: a destination overlaps a source or the other destination");

  // ---- once per device: the device address of the static plan ----
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return fail(FCG_ERR_CUDA, "cudaGetDevice: %s", cudaGetErrorString(e));
  if (dev < 0 || dev >= MAX_DEVICES) return fail(FCG_ERR_INVALID_ARG, "fcg_segment_shift_static: device ordinal %d beyond %d", dev, MAX_DEVICES - 1);
  unsigned char *plan = nullptr;
  {
    std::lock_guard<std::mutex> lk(g_mu);
    if (!g_plan_dev[dev]) {
      void *p = nullptr;
      e = cudaGetSymbolAddress(&p, g_static_plan);        // resolved for the CURRENT device, which is `dev`
      if (e != cudaSuccess || !p) return fail(FCG_ERR_CUDA, "cudaGetSymbolAddress(g_static_plan) on device %d: %s", dev, cudaGetErrorString(e));
      g_plan_dev[dev] = static_cast<unsigned char *>(p);
    }
    plan = g_plan_dev[dev];
  }

  // ---- the plan of this call ----
  PlanArgs a;
  memset(&a, 0, sizeof a);
  const bool rotate = rope_mode != FCG_ROPE_NONE && delta != 0;
  a.entry.k_src = (uint64_t)(uintptr_t)k_src;
  a.entry.v_src = (uint64_t)(uintptr_t)v_src;
  a.entry.k_dst = (uint64_t)(uintptr_t)k_dst;
  a.entry.v_dst = (uint64_t)(uintptr_t)v_dst;
  a.entry.src_layer_stride = a.entry.dst_layer_stride = (int64_t)n_kv_heads * n_tokens;
  a.entry.src_head_stride = a.entry.dst_head_stride = n_tokens;
  a.entry.table_off = rotate ? 0 : -1;
  a.n_tokens = n_tokens;
  a.n_table = rotate ? head_dim / 2 : 0;
  for (int j = 0; j < a.n_table; ++j) {
    const double theta = inv_freq ? inv_freq[j] : pow(rope_base, -2.0 * (double)j / (double)head_dim);
    const double phi = (double)delta * theta;
    split(cos(phi), a.table[j].x, a.table[j].y);
    split(sin(phi), a.table[j].z, a.table[j].w);
  }

  cudaStream_t s = static_cast<cudaStream_t>(stream);
  const int n_chunks = (n_tokens + CHUNK_TOKENS - 1) / CHUNK_TOKENS;
  const int work = n_chunks > MAX_HALF ? n_chunks : MAX_HALF;
  static_plan_kernel<<<(work + 255) / 256, 256, 0, s>>>(a);
  e = cudaGetLastError();
  if (e != cudaSuccess) return fail(FCG_ERR_CUDA, "static_plan_kernel: %s", cudaGetErrorString(e));

  fcg::StitchParams sp;
  sp.any_fp8 = 0;
  sp.entries = reinterpret_cast<const fcg::StitchEntryDev *>(plan + OFF_ENTRY);
  sp.chunks = reinterpret_cast<const fcg::StitchChunkDev *>(plan + OFF_CHUNKS);
  sp.table = reinterpret_cast<const float4 *>(plan + OFF_TABLE);
  sp.n_chunks = n_chunks;
  sp.n_layers = n_layers;
  sp.n_kv_heads = n_kv_heads;
  sp.interleaved = rope_mode == FCG_ROPE_INTERLEAVED ? 1 : 0;
  sp.head_dim = head_dim;
  e = fcg::launch_stitch(sp, head_dim, s);
  if (e != cudaSuccess) return fail(FCG_ERR_CUDA, "launch_stitch: %s", cudaGetErrorString(e));
  return FCG_OK;
}

}  // extern "C"
