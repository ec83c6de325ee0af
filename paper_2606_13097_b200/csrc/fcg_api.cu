// Host side of libfcg.so: the C ABI of include/fcg.h -- segment library (S1), stitch-plan builder and
// page allocator (S2), and the launch logic for S3-S6.  Everything here is integer bookkeeping plus
// the fp64 evaluation of the per-entry RoPE table; all K/V/q arithmetic runs in the kernels.
#include <cuda.h>   // CUtensorMap types only: the driver entry point is resolved at run time, libcuda is not linked
#include <cuda_runtime.h>
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <string.h>

#include <algorithm>
#include <map>
#include <string>
#include <vector>

#include "../../include/fcg.h"
#include "fcg_internal.h"

namespace {

thread_local std::string g_err = "";

fcg_status_t fail(fcg_status_t st, const char *fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  g_err = buf;
  return st;
}

#define FCG_CUDA(expr)                                                                         \
  do {                                                                                         \
    cudaError_t e__ = (expr);                                                                  \
    if (e__ != cudaSuccess) return fail(FCG_ERR_CUDA, "%s: %s", #expr, cudaGetErrorString(e__)); \
  } while (0)

constexpr uint64_t ALIGN = 256;
constexpr int BLOB_SLOTS = 16;
constexpr uint64_t BLOB_BYTES = 1ull << 20;
constexpr int KV_TILE = 64;          // tokens per attention tile (fcg_attn_split.cu BN)

uint64_t align_up(uint64_t x, uint64_t a = ALIGN) { return (x + a - 1) / a * a; }

struct SegmentRec {
  bool live = false;
  uint64_t offset = 0, bytes = 0;   // in the arena (resident) or in the host tier (offloaded); K then V
  bool resident = true;
  int32_t n_tokens = 0, orig_start = 0;
  int32_t fmt = FCG_STORE_BF16;     // FCG_STORE_FP8_E4M3: K codes, K scale bytes, V codes, V scale bytes (R26)
};

struct TaskRec {
  bool live = false;
  uint32_t gen = 0;                 // bumped when the task is stitched or released (validates patch plans)
  std::vector<int32_t> pages;
  int32_t capacity = 0, n_tokens = 0;
  std::vector<uint8_t> filled;
  int32_t filled_prefix = 0;        // every x < filled_prefix is filled
  std::vector<std::pair<int32_t, int32_t>> spans;   // (dst_offset, n_tokens) of the stitched entries, plan order
};

struct BlobSlot {
  unsigned char *host = nullptr;    // pinned
  unsigned char *dev = nullptr;     // inside the workspace
  cudaEvent_t ev = nullptr;
  bool in_flight = false;
  uint64_t gen = 0;                 // bumped at every acquisition (validates the cached patch blob)
};

struct FreeRange {
  uint64_t off, bytes;
};

}  // namespace

namespace fcg {
// for the other translation units of the library (fcg_static.cu): the message fcg_last_error() returns on this thread
void set_last_error(const char *msg) { g_err = msg ? msg : ""; }
}  // namespace fcg

struct fcg_patch_plan;
extern "C++" __attribute__((visibility("hidden"))) void free_plans(struct fcg_library *lib);

struct fcg_library {
  fcg_config_t cfg;
  std::vector<double> inv_freq;
  unsigned char *arena = nullptr;
  uint64_t k_pool_off = 0, v_pool_off = 0, pool_bytes = 0, table_off = 0, ws_off = 0, seg_off = 0, seg_bytes = 0;
  uint64_t scratch_off = 0, scratch_bytes = 0;   // workspace after the blob slots
  uint64_t scratch_total = 0;                    // scratch_bytes as created (the host variants shrink scratch_bytes for the duration of a call)
  int32_t pages_per_task = 0;
  std::vector<int32_t> page_stack;               // LIFO: back() is handed out next
  std::vector<SegmentRec> segments;
  std::vector<FreeRange> seg_free;               // sorted by offset
  unsigned char *host_arena = nullptr;           // second tier: pinned host memory (Eq. 3), NULL if none
  unsigned char *host_dev = nullptr;             // the same memory as the device sees it (zero-copy stitch)
  std::vector<FreeRange> host_free;              // offsets relative to host_arena, sorted
  std::vector<TaskRec> tasks;
  BlobSlot slots[BLOB_SLOTS];
  // fcg_patch_host: the host->device copies run on the library's own stream, ordered after the last patch call
  // (the staging area belongs to patch calls only), so they overlap a stitch enqueued just before on the caller's stream
  cudaStream_t copy_stream = nullptr, d2h_stream = nullptr;
  static constexpr int HOST_GROUPS = 4;          // layer groups of a host call: copy in / attend / copy out pipelined
  cudaEvent_t h2d_ev[HOST_GROUPS] = {}, attn_ev[HOST_GROUPS] = {}, d2h_ev = nullptr;
  // DESIGN.md R29: scratch area, plan blobs and recycled pages are library-wide, so a call issued on another stream than
  // the previous call first waits for that call's device work (last_ev, recorded at the end of every enqueueing call)
  cudaEvent_t last_ev = nullptr;
  cudaStream_t last_stream = nullptr;
  bool have_last = false;
  int n_sms = 148;                               // SMs of cfg.device (split selection)
  uint32_t task_gen = 0;
  // the plan blob of the last patch call: a call that produces the same bytes (the same patch issued for the next layer)
  // reuses the copy that is already on the device instead of uploading it again
  std::vector<unsigned char> patch_blob_copy;
  int patch_blob_slot = -1;
  uint64_t patch_blob_gen = 0;
  cudaStream_t patch_blob_stream = nullptr;      // the stream that uploaded it (reuse only on the same stream)
  cudaEvent_t prefetch_ev = nullptr;             // fcg_stitch_prefetch: the host->device copies of one call have landed
  cudaEvent_t staging_ev = nullptr;              // last use of the host-call staging area
  bool have_staging_ev = false;
  std::vector<unsigned char> dry_blob;           // host scratch of dry_check_patch
  int n_plans_live = 0;
  std::vector<struct fcg_patch_plan *> plans;    // live patch plans (freed by fcg_library_destroy if the caller did not)
  int next_slot = 0;
  fcg_stats_t stats;
  int n_segments_live = 0, n_tasks_live = 0;
  int32_t tc_min_rows = 1;                       // rows per kv head from which the tcgen05 path is used
  fcg::TmaDesc tm_k, tm_v;                       // K / V pool tensor maps for the tcgen05 path
  bool have_tma = false;
  int32_t force_splits = 0;                      // > 0: KV splits per task (clamped to its tile count); 0 = choose_splits
  bool mix_classes = false;                      // a batch with several CTA classes as ONE interleaved launch (head_dim 128) instead of one per class
  bool use_pairs = false;                        // > 128 rows per kv head at head_dim 128: CTA pairs (cta_group::2) instead of two Q tiles per CTA

  uint16_t *k_pool() const { return reinterpret_cast<uint16_t *>(arena + k_pool_off); }
  uint16_t *v_pool() const { return reinterpret_cast<uint16_t *>(arena + v_pool_off); }
  int32_t *tables() const { return reinterpret_cast<int32_t *>(arena + table_off); }
  uint64_t kv_row_bytes() const { return (uint64_t)cfg.head_dim * 2; }
  uint64_t seg_bytes_for(int64_t n, int32_t fmt = FCG_STORE_BF16) const {
    const uint64_t rows = (uint64_t)cfg.n_layers * cfg.n_kv_heads * (uint64_t)n;
    if (fmt == FCG_STORE_FP8_E4M3) return 2 * (fp8_code_bytes(n) + align_up(rows));
    return 2 * align_up(rows * kv_row_bytes());
  }
  uint64_t fp8_code_bytes(int64_t n) const { return align_up((uint64_t)cfg.n_layers * cfg.n_kv_heads * (uint64_t)n * cfg.head_dim); }
};

namespace {

bool geometry_ok(const fcg_config_t *c) {
  if (!c) return false;
  if (c->n_layers <= 0 || c->n_kv_heads <= 0 || c->n_q_heads <= 0 || c->n_q_heads % c->n_kv_heads) return false;
  if (c->n_layers > 65535 || c->n_kv_heads > 65535) return false;      // layers / kv heads run along grid y
  if (c->head_dim < 16 || c->head_dim > 256 || c->head_dim % 16) return false;      // R27
  if (c->page_size != 8 && c->page_size != 16 && c->page_size != 32 && c->page_size != 64) return false;
  if (c->rope_mode != FCG_ROPE_NONE && c->rope_mode != FCG_ROPE_HALF_SPLIT && c->rope_mode != FCG_ROPE_INTERLEAVED) return false;
  if (c->rope_mode != FCG_ROPE_NONE && !c->inv_freq && !(c->rope_base > 0.0)) return false;
  if (c->max_segments <= 0 || c->max_tasks <= 0 || c->max_task_tokens <= 0 || c->n_pages == 0) return false;
  return true;
}

struct Layout {
  uint64_t k_pool_off, v_pool_off, pool_bytes, table_off, ws_off, ws_bytes, seg_off;
  int32_t pages_per_task;
};

Layout layout_of(const fcg_config_t *c) {
  Layout l;
  l.pool_bytes = align_up((uint64_t)c->n_layers * c->n_pages * c->n_kv_heads * c->page_size * c->head_dim * 2);
  l.k_pool_off = 0;
  l.v_pool_off = l.pool_bytes;
  l.table_off = 2 * l.pool_bytes;
  l.pages_per_task = (c->max_task_tokens + c->page_size - 1) / c->page_size;
  l.ws_off = l.table_off + align_up((uint64_t)c->max_tasks * l.pages_per_task * 4);
  l.ws_bytes = align_up(c->workspace_bytes ? c->workspace_bytes : (256ull << 20));
  l.seg_off = l.ws_off + l.ws_bytes;
  return l;
}

// TMA tensor map of one pool [L][n_pages][Hkv][P][D] bf16 as the 5-D tensor (D, P, Hkv, n_pages, L), innermost
// first; box = (64 columns, one page, 1, 1, 1) with 128B swizzle = one 64-column half of one head's page slice,
// which lands in shared memory exactly in the K-major / MN-major UMMA operand layout (fcg_attn_tc.cu).
fcg_status_t make_pool_tensor_map(const fcg_config_t &c, void *pool, fcg::TmaDesc *out) {
  typedef CUresult (*encode_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
  static encode_fn encode = nullptr;
  if (!encode) {
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    FCG_CUDA(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres));
    if (!fn || qres != cudaDriverEntryPointSuccess) return fail(FCG_ERR_CUDA, "cuTensorMapEncodeTiled is not available in this driver");
    encode = reinterpret_cast<encode_fn>(fn);
  }
  static_assert(sizeof(CUtensorMap) == sizeof(fcg::TmaDesc), "CUtensorMap is 128 bytes");
  const cuuint64_t D = c.head_dim, P = c.page_size, H = c.n_kv_heads;
  const cuuint64_t dims[5] = {D, P, H, c.n_pages, (cuuint64_t)c.n_layers};
  const cuuint64_t strides[4] = {D * 2, P * D * 2, H * P * D * 2, (cuuint64_t)c.n_pages * H * P * D * 2};
  const cuuint32_t box[5] = {64, (cuuint32_t)P, 1, 1, 1};
  const cuuint32_t estr[5] = {1, 1, 1, 1, 1};
  CUresult r = encode(reinterpret_cast<CUtensorMap *>(out), CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 5, pool, dims, strides, box, estr,
                      CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                      CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return fail(FCG_ERR_CUDA, "cuTensorMapEncodeTiled failed with CUresult %d", (int)r);
  return FCG_OK;
}

// Every API call runs with the library's device current and puts the caller's device back on return.
struct DeviceGuard {
  int prev = -1;
  bool changed = false;
  cudaError_t err;
  explicit DeviceGuard(int dev) {
    err = cudaGetDevice(&prev);
    if (err == cudaSuccess && prev != dev) {
      err = cudaSetDevice(dev);
      changed = err == cudaSuccess;
    }
  }
  ~DeviceGuard() {
    if (changed) cudaSetDevice(prev);
  }
};
#define FCG_DEVICE(lib)                \
  DeviceGuard dg__((lib)->cfg.device); \
  if (dg__.err != cudaSuccess) return fail(FCG_ERR_CUDA, "cudaSetDevice(%d): %s", (lib)->cfg.device, cudaGetErrorString(dg__.err))

// R29: order this call after the previous call's device work when the stream changes.  A capturing stream takes
// no part in it (events recorded inside a capture cannot be waited for outside): only fcg_patch_planned may be
// captured, and the caller orders the graph against other work on the library.
fcg_status_t order_after_previous(fcg_library *lib, cudaStream_t stream, bool *capturing) {
  cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
  if (cudaStreamIsCapturing(stream, &cs) != cudaSuccess) {
    cudaGetLastError();
    cs = cudaStreamCaptureStatusNone;
  }
  *capturing = cs != cudaStreamCaptureStatusNone;
  if (!*capturing && lib->have_last && stream != lib->last_stream) FCG_CUDA(cudaStreamWaitEvent(stream, lib->last_ev, 0));
  return FCG_OK;
}
fcg_status_t mark_last(fcg_library *lib, cudaStream_t stream) {
  FCG_CUDA(cudaEventRecord(lib->last_ev, stream));
  lib->last_stream = stream;
  lib->have_last = true;
  return FCG_OK;
}
// calls that upload a plan blob from pinned host memory cannot be captured into a CUDA graph (a replay would re-read
// host memory that has been reused since)
#define FCG_ORDER(lib, stream)                                                                                          \
  do {                                                                                                                  \
    bool cap__ = false;                                                                                                 \
    fcg_status_t st__ = order_after_previous((lib), (stream), &cap__);                                                  \
    if (st__ != FCG_OK) return st__;                                                                                    \
    if (cap__)                                                                                                          \
      return fail(FCG_ERR_INVALID_ARG, "this call cannot be captured into a CUDA graph (it uploads a plan blob): use "   \
                                       "fcg_patch_plan_create + fcg_patch_planned");                                    \
  } while (0)

// A blob slot in use by one call: whatever path the call leaves by, once anything that reads the slot has been
// enqueued the slot's event is recorded, so the pinned blob is not rewritten under a copy in flight.
struct SlotUse {
  BlobSlot *slot = nullptr;
  cudaStream_t stream = nullptr;
  bool enqueued = false;
  ~SlotUse() {
    if (slot && enqueued && cudaEventRecord(slot->ev, stream) == cudaSuccess) slot->in_flight = true;
  }
};

// acquire a blob slot whose previous consumer kernels have finished
fcg_status_t acquire_slot(fcg_library *lib, BlobSlot **out) {
  BlobSlot &s = lib->slots[lib->next_slot];
  lib->next_slot = (lib->next_slot + 1) % BLOB_SLOTS;
  if (s.in_flight) {
    FCG_CUDA(cudaEventSynchronize(s.ev));
    s.in_flight = false;
  }
  s.gen++;
  *out = &s;
  return FCG_OK;
}

struct BlobWriter {
  unsigned char *base;
  uint64_t used = 0, cap;
  BlobWriter(unsigned char *b, uint64_t c) : base(b), cap(c) {}
  // returns the byte offset of `bytes` reserved bytes (16-byte aligned) or UINT64_MAX
  uint64_t reserve(uint64_t bytes) {
    uint64_t off = align_up(used, 16);
    if (off + bytes > cap) return UINT64_MAX;
    used = off + bytes;
    return off;
  }
};

// first-fit over a sorted free list; returns the index of the range or free_list.size()
size_t range_find(const std::vector<FreeRange> &fl, uint64_t bytes) {
  for (size_t i = 0; i < fl.size(); ++i)
    if (fl[i].bytes >= bytes) return i;
  return fl.size();
}
void range_take(std::vector<FreeRange> &fl, size_t i, uint64_t bytes) {
  if (fl[i].bytes == bytes)
    fl.erase(fl.begin() + i);
  else {
    fl[i].off += bytes;
    fl[i].bytes -= bytes;
  }
}
// insert and coalesce with the neighbours
void range_give(std::vector<FreeRange> &fl, uint64_t off, uint64_t bytes) {
  FreeRange fr{off, bytes};
  auto it = std::lower_bound(fl.begin(), fl.end(), fr, [](const FreeRange &a, const FreeRange &b) { return a.off < b.off; });
  it = fl.insert(it, fr);
  if (it + 1 != fl.end() && it->off + it->bytes == (it + 1)->off) {
    it->bytes += (it + 1)->bytes;
    fl.erase(it + 1);
  }
  if (it != fl.begin() && (it - 1)->off + (it - 1)->bytes == it->off) {
    (it - 1)->bytes += it->bytes;
    fl.erase(it);
  }
}

// lowest free segment id and first-fit arena range for an n-token segment; nothing changes until commit
struct SegmentSlot {
  int32_t sid = -1;
  size_t fi = 0;
  uint64_t off = 0, bytes = 0;
};

fcg_status_t find_segment_slot(fcg_library *lib, int32_t n_tokens, SegmentSlot &sl, int32_t fmt = FCG_STORE_BF16) {
  const fcg_config_t &c = lib->cfg;
  sl.sid = -1;
  for (int32_t i = 0; i < c.max_segments; ++i)
    if (!lib->segments[i].live) {
      sl.sid = i;
      break;
    }
  if (sl.sid < 0) return fail(FCG_ERR_OUT_OF_ARENA, "segment table full (%d)", c.max_segments);
  sl.bytes = lib->seg_bytes_for(n_tokens, fmt);
  sl.fi = range_find(lib->seg_free, sl.bytes);
  if (sl.fi == lib->seg_free.size())
    return fail(FCG_ERR_OUT_OF_ARENA, "no free arena range of %llu bytes for a %d-token segment", (unsigned long long)sl.bytes, n_tokens);
  sl.off = lib->seg_free[sl.fi].off;
  return FCG_OK;
}

void commit_segment_slot(fcg_library *lib, const SegmentSlot &sl, int32_t n_tokens, int32_t orig_start, int32_t fmt = FCG_STORE_BF16) {
  range_take(lib->seg_free, sl.fi, sl.bytes);
  SegmentRec &s = lib->segments[sl.sid];
  s.live = true;
  s.fmt = fmt;
  s.offset = sl.off;
  s.bytes = sl.bytes;
  s.n_tokens = n_tokens;
  s.orig_start = orig_start;
  s.resident = true;
  lib->n_segments_live++;
}

// Host side of one launch of the gather + RoPE-shift kernel (S3): entries, chunks, the per-delta cos/sin table
// and the page ids that go into page tables, packed into one pinned blob and shipped with one async H2D.
struct GatherBuilder {
  std::vector<fcg::StitchEntryDev> entries;
  std::vector<fcg::StitchChunkDev> chunks;
  std::vector<float4> table;
  std::vector<int32_t> pages;                    // page ids, copied device-to-device into page tables after the H2D
  std::map<int32_t, int32_t> table_of_delta;
  bool any_fp8 = false;

  // first float4 of the table of `delta`, or -1 for a bit copy
  int32_t table_for(const fcg_library *lib, int32_t delta) {
    if (lib->cfg.rope_mode == FCG_ROPE_NONE || delta == 0) return -1;
    auto it = table_of_delta.find(delta);
    if (it != table_of_delta.end()) return it->second;
    const int half = lib->cfg.head_dim / 2;
    const int32_t off = (int32_t)table.size();
    table_of_delta[delta] = off;
    for (int j = 0; j < half; ++j) {
      const double phi = (double)delta * lib->inv_freq[j];
      const double cs = cos(phi), sn = sin(phi);
      // hi part: 16 significant bits, so that (bf16 x hi) is exact in fp32; lo: the remainder
      auto split = [](double x, float &hi, float &lo) {
        float f = (float)x;
        uint32_t b;
        memcpy(&b, &f, 4);
        b = (b + 0x80u) & 0xffffff00u;
        memcpy(&hi, &b, 4);
        lo = (float)(x - (double)hi);
      };
      float4 t;
      split(cs, t.x, t.y);
      split(sn, t.z, t.w);
      table.push_back(t);
    }
    return off;
  }

  // row-space descriptors (fcg_internal.h)
  void pool_side(const fcg_library *lib, uint64_t &k, uint64_t &v, int64_t &layer_stride, int32_t &head_stride) const {
    const fcg_config_t &c = lib->cfg;
    k = (uint64_t)(uintptr_t)lib->k_pool();
    v = (uint64_t)(uintptr_t)lib->v_pool();
    layer_stride = (int64_t)c.n_pages * c.n_kv_heads * c.page_size;
    head_stride = c.page_size;
  }
  void segment_side(const fcg_library *lib, const unsigned char *tier_base, uint64_t off, uint64_t bytes, int32_t n,
                    uint64_t &k, uint64_t &v, int64_t &layer_stride, int32_t &head_stride) const {
    k = (uint64_t)(uintptr_t)(tier_base + off);
    v = (uint64_t)(uintptr_t)(tier_base + off + bytes / 2);
    layer_stride = (int64_t)lib->cfg.n_kv_heads * n;
    head_stride = n;
  }
  // source side of an entry that reads a library segment (either tier, either storage format)
  void source_segment(const fcg_library *lib, const SegmentRec &s, fcg::StitchEntryDev &de) {
    segment_side(lib, s.resident ? lib->arena : lib->host_dev, s.offset, s.bytes, s.n_tokens, de.k_src, de.v_src, de.src_layer_stride,
                 de.src_head_stride);
    de.src_fp8 = s.fmt == FCG_STORE_FP8_E4M3 ? 1 : 0;
    de.k_exp = de.v_exp = 0;
    if (de.src_fp8) {
      de.k_exp = de.k_src + lib->fp8_code_bytes(s.n_tokens);
      de.v_exp = de.v_src + lib->fp8_code_bytes(s.n_tokens);
      any_fp8 = true;
    }
  }
  int32_t pool_tok(const fcg_library *lib, int32_t page, int32_t slot) const {
    return page * lib->cfg.n_kv_heads * lib->cfg.page_size + slot;
  }
  uint64_t blob_bytes() const {
    return align_up(entries.size() * sizeof(fcg::StitchEntryDev), 16) + align_up(chunks.size() * sizeof(fcg::StitchChunkDev), 16) +
           align_up(pages.size() * sizeof(int32_t), 16) + table.size() * sizeof(float4);
  }
};

struct GatherBlob {
  SlotUse use;
  BlobSlot *slot = nullptr;
  uint64_t off_pages = 0;
};

// pack the builder into a blob slot, ship it, launch the kernel; page ids sit at out.off_pages of the slot.  The
// slot's event is recorded when `out` goes out of scope (SlotUse), after whatever else the caller enqueues from it.
fcg_status_t enqueue_gather(fcg_library *lib, const GatherBuilder &gb, cudaStream_t stream, GatherBlob &out) {
  const fcg_config_t &c = lib->cfg;
  if (gb.blob_bytes() > BLOB_BYTES) return fail(FCG_ERR_OUT_OF_ARENA, "plan blob of %llu bytes exceeds %llu", (unsigned long long)gb.blob_bytes(), (unsigned long long)BLOB_BYTES);
  if ((uint64_t)c.n_pages * c.n_kv_heads * c.page_size > 0x7fffffffull) return fail(FCG_ERR_INVALID_ARG, "pool too large for 32-bit row offsets");
  BlobSlot *slot = nullptr;
  fcg_status_t st = acquire_slot(lib, &slot);
  if (st != FCG_OK) return st;
  out.use.slot = slot;
  out.use.stream = stream;
  BlobWriter bw(slot->host, BLOB_BYTES);
  const uint64_t off_entries = bw.reserve(gb.entries.size() * sizeof(fcg::StitchEntryDev));
  const uint64_t off_chunks = bw.reserve(gb.chunks.size() * sizeof(fcg::StitchChunkDev));
  const uint64_t off_pages = bw.reserve(gb.pages.size() * sizeof(int32_t));
  const uint64_t off_table = bw.reserve(gb.table.size() * sizeof(float4));
  if (!gb.entries.empty()) memcpy(slot->host + off_entries, gb.entries.data(), gb.entries.size() * sizeof(fcg::StitchEntryDev));
  if (!gb.chunks.empty()) memcpy(slot->host + off_chunks, gb.chunks.data(), gb.chunks.size() * sizeof(fcg::StitchChunkDev));
  if (!gb.pages.empty()) memcpy(slot->host + off_pages, gb.pages.data(), gb.pages.size() * sizeof(int32_t));
  if (!gb.table.empty()) memcpy(slot->host + off_table, gb.table.data(), gb.table.size() * sizeof(float4));
  if (bw.used > 0) {
    FCG_CUDA(cudaMemcpyAsync(slot->dev, slot->host, bw.used, cudaMemcpyHostToDevice, stream));
    out.use.enqueued = true;
  }
  fcg::StitchParams sp;
  sp.entries = reinterpret_cast<const fcg::StitchEntryDev *>(slot->dev + off_entries);
  sp.chunks = reinterpret_cast<const fcg::StitchChunkDev *>(slot->dev + off_chunks);
  sp.table = reinterpret_cast<const float4 *>(slot->dev + off_table);
  sp.any_fp8 = gb.any_fp8 ? 1 : 0;
  sp.n_chunks = (int32_t)gb.chunks.size();
  sp.n_layers = c.n_layers;
  sp.n_kv_heads = c.n_kv_heads;
  sp.interleaved = c.rope_mode == FCG_ROPE_INTERLEAVED ? 1 : 0;
  sp.head_dim = c.head_dim;
  if (!gb.chunks.empty()) {
    FCG_CUDA(fcg::launch_stitch(sp, c.head_dim, stream));
    lib->stats.stitch_launches++;
  }
  out.slot = slot;
  out.off_pages = off_pages;
  return FCG_OK;
}

}  // namespace

extern "C" {

const char *fcg_last_error(void) { return g_err.c_str(); }
const char *fcg_version(void) { return "0.1.0 sm_100a"; }

uint64_t fcg_arena_bytes_required(const fcg_config_t *cfg, uint64_t segment_tokens) {
  if (!geometry_ok(cfg)) return 0;
  Layout l = layout_of(cfg);
  const uint64_t per_tok = (uint64_t)cfg->n_layers * cfg->n_kv_heads * cfg->head_dim * 2 * 2;
  return l.seg_off + segment_tokens * per_tok + (uint64_t)cfg->max_segments * 2 * ALIGN + 4096;
}

fcg_status_t fcg_library_create(const fcg_config_t *cfg, fcg_library_t **out) {
  if (!out) return fail(FCG_ERR_INVALID_ARG, "out is NULL");
  *out = nullptr;
  if (!geometry_ok(cfg))
    return fail(FCG_ERR_INVALID_ARG,
                "bad configuration (head_dim must be a multiple of 16 in [16, 256], page_size 8/16/32/64, n_q_heads %% n_kv_heads == 0, "
                "capacities > 0)");
  if (!cfg->arena || ((uintptr_t)cfg->arena % ALIGN)) return fail(FCG_ERR_INVALID_ARG, "arena must be a 256-byte aligned device pointer");
  Layout l = layout_of(cfg);
  if (l.ws_bytes < (uint64_t)BLOB_SLOTS * BLOB_BYTES + (16ull << 20))
    return fail(FCG_ERR_INVALID_ARG, "workspace_bytes must be at least %llu", (unsigned long long)((uint64_t)BLOB_SLOTS * BLOB_BYTES + (16ull << 20)));
  if (l.seg_off > cfg->arena_bytes)
    return fail(FCG_ERR_OUT_OF_ARENA, "arena of %llu bytes cannot hold pools + tables + workspace (%llu bytes)",
                (unsigned long long)cfg->arena_bytes, (unsigned long long)l.seg_off);
  int n_dev = 0;
  FCG_CUDA(cudaGetDeviceCount(&n_dev));
  if (cfg->device < 0 || cfg->device >= n_dev) return fail(FCG_ERR_INVALID_ARG, "device %d out of range", cfg->device);
  DeviceGuard dg(cfg->device);
  if (dg.err != cudaSuccess) return fail(FCG_ERR_CUDA, "cudaSetDevice(%d): %s", cfg->device, cudaGetErrorString(dg.err));

  fcg_library *lib = new fcg_library();
  lib->cfg = *cfg;
  if (cudaDeviceGetAttribute(&lib->n_sms, cudaDevAttrMultiProcessorCount, cfg->device) != cudaSuccess || lib->n_sms <= 0) {
    cudaGetLastError();
    lib->n_sms = 148;
  }
  lib->cfg.workspace_bytes = l.ws_bytes;
  const int half = cfg->head_dim / 2;
  lib->inv_freq.resize(half);
  for (int j = 0; j < half; ++j)
    lib->inv_freq[j] = cfg->inv_freq ? cfg->inv_freq[j] : pow(cfg->rope_base, -2.0 * (double)j / (double)cfg->head_dim);
  lib->cfg.inv_freq = nullptr;
  lib->arena = static_cast<unsigned char *>(cfg->arena);
  lib->k_pool_off = l.k_pool_off;
  lib->v_pool_off = l.v_pool_off;
  lib->pool_bytes = l.pool_bytes;
  lib->table_off = l.table_off;
  lib->ws_off = l.ws_off;
  lib->seg_off = l.seg_off;
  lib->seg_bytes = cfg->arena_bytes - l.seg_off;
  lib->pages_per_task = l.pages_per_task;
  lib->scratch_off = l.ws_off + (uint64_t)BLOB_SLOTS * BLOB_BYTES;
  lib->scratch_bytes = l.ws_bytes - (uint64_t)BLOB_SLOTS * BLOB_BYTES;
  lib->scratch_total = lib->scratch_bytes;
  lib->page_stack.resize(cfg->n_pages);
  for (uint32_t i = 0; i < cfg->n_pages; ++i) lib->page_stack[i] = (int32_t)(cfg->n_pages - 1 - i);  // back() == 0
  lib->segments.resize(cfg->max_segments);
  lib->tasks.resize(cfg->max_tasks);
  if (lib->seg_bytes) lib->seg_free.push_back({lib->seg_off, lib->seg_bytes});
  memset(&lib->stats, 0, sizeof lib->stats);
  for (int i = 0; i < BLOB_SLOTS; ++i) {
    cudaError_t e = cudaHostAlloc((void **)&lib->slots[i].host, BLOB_BYTES, cudaHostAllocDefault);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&lib->slots[i].ev, cudaEventDisableTiming);
    if (e != cudaSuccess) {
      for (int j = 0; j <= i; ++j) {
        if (lib->slots[j].host) cudaFreeHost(lib->slots[j].host);
        if (lib->slots[j].ev) cudaEventDestroy(lib->slots[j].ev);
      }
      delete lib;
      return fail(FCG_ERR_CUDA, "blob slot allocation: %s", cudaGetErrorString(e));
    }
    lib->slots[i].dev = lib->arena + l.ws_off + (uint64_t)i * BLOB_BYTES;
  }
  {
    cudaError_t e = cudaStreamCreateWithFlags(&lib->copy_stream, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&lib->d2h_stream, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&lib->last_ev, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&lib->staging_ev, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&lib->prefetch_ev, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&lib->d2h_ev, cudaEventDisableTiming);
    for (int g = 0; g < fcg_library::HOST_GROUPS && e == cudaSuccess; ++g) {
      e = cudaEventCreateWithFlags(&lib->h2d_ev[g], cudaEventDisableTiming);
      if (e == cudaSuccess) e = cudaEventCreateWithFlags(&lib->attn_ev[g], cudaEventDisableTiming);
    }
    if (e != cudaSuccess) {
      fcg_library_destroy(lib);
      return fail(FCG_ERR_CUDA, "copy stream / events: %s", cudaGetErrorString(e));
    }
  }
  if (cfg->host_arena && cfg->host_arena_bytes) {
    cudaPointerAttributes attr;
    cudaError_t e = cudaPointerGetAttributes(&attr, cfg->host_arena);
    if (e != cudaSuccess || attr.type != cudaMemoryTypeHost || !attr.devicePointer || ((uintptr_t)cfg->host_arena % ALIGN)) {
      cudaGetLastError();
      fcg_library_destroy(lib);
      return fail(FCG_ERR_INVALID_ARG, "host_arena must be pinned (cudaHostAlloc / cudaHostRegister) and 256-byte aligned");
    }
    lib->host_arena = static_cast<unsigned char *>(cfg->host_arena);
    lib->host_dev = static_cast<unsigned char *>(attr.devicePointer);
    lib->host_free.push_back({0, cfg->host_arena_bytes / ALIGN * ALIGN});
  }
  {
    fcg_status_t st = make_pool_tensor_map(lib->cfg, lib->k_pool(), &lib->tm_k);
    if (st == FCG_OK) st = make_pool_tensor_map(lib->cfg, lib->v_pool(), &lib->tm_v);
    if (st != FCG_OK) {
      fcg_library_destroy(lib);
      return st;
    }
    lib->have_tma = true;
  }
  *out = lib;
  return FCG_OK;
}

fcg_status_t fcg_library_destroy(fcg_library_t *lib) {
  if (!lib) return fail(FCG_ERR_INVALID_ARG, "lib is NULL");
  DeviceGuard dg(lib->cfg.device);
  cudaDeviceSynchronize();
  for (int i = 0; i < BLOB_SLOTS; ++i) {
    if (lib->slots[i].host) cudaFreeHost(lib->slots[i].host);
    if (lib->slots[i].ev) cudaEventDestroy(lib->slots[i].ev);
  }
  free_plans(lib);
  if (lib->copy_stream) cudaStreamDestroy(lib->copy_stream);
  if (lib->d2h_stream) cudaStreamDestroy(lib->d2h_stream);
  if (lib->last_ev) cudaEventDestroy(lib->last_ev);
  if (lib->staging_ev) cudaEventDestroy(lib->staging_ev);
  if (lib->prefetch_ev) cudaEventDestroy(lib->prefetch_ev);
  if (lib->d2h_ev) cudaEventDestroy(lib->d2h_ev);
  for (int g = 0; g < fcg_library::HOST_GROUPS; ++g) {
    if (lib->h2d_ev[g]) cudaEventDestroy(lib->h2d_ev[g]);
    if (lib->attn_ev[g]) cudaEventDestroy(lib->attn_ev[g]);
  }
  delete lib;
  return FCG_OK;
}

// ------------------------------------------------------------------------------------------ S1
fcg_status_t fcg_segment_register(fcg_library_t *lib, const void *k, const void *v, int32_t n_tokens,
                                  int32_t orig_start, const int64_t *strides, void *stream, int32_t *seg_id_out) {
  if (!lib || !k || !v || !seg_id_out) return fail(FCG_ERR_INVALID_ARG, "NULL argument");
  if (n_tokens <= 0 || orig_start < 0) return fail(FCG_ERR_INVALID_ARG, "n_tokens must be > 0 and orig_start >= 0");
  const fcg_config_t &c = lib->cfg;
  int64_t st[4] = {(int64_t)c.n_kv_heads * n_tokens * c.head_dim, (int64_t)n_tokens * c.head_dim, c.head_dim, 1};
  if (strides) {
    if (strides[3] != 1) return fail(FCG_ERR_INVALID_ARG, "strides[3] must be 1 (contiguous head_dim)");
    for (int i = 0; i < 3; ++i) {
      if (strides[i] % 8) return fail(FCG_ERR_INVALID_ARG, "strides must be multiples of 8 elements (16-byte rows)");
      st[i] = strides[i];
    }
  }
  if (((uintptr_t)k % 16) || ((uintptr_t)v % 16)) return fail(FCG_ERR_INVALID_ARG, "k and v must be 16-byte aligned");
  SegmentSlot sl;
  fcg_status_t sst = find_segment_slot(lib, n_tokens, sl);
  if (sst != FCG_OK) return sst;
  const int32_t sid = sl.sid;
  const uint64_t off = sl.off, bytes = sl.bytes;

  fcg::RegisterParams rp;
  rp.k_src = static_cast<const uint16_t *>(k);
  rp.v_src = static_cast<const uint16_t *>(v);
  rp.k_dst = reinterpret_cast<uint16_t *>(lib->arena + off);
  rp.v_dst = reinterpret_cast<uint16_t *>(lib->arena + off + bytes / 2);
  rp.s_layer = st[0];
  rp.s_head = st[1];
  rp.s_tok = st[2];
  rp.n_layers = c.n_layers;
  rp.n_kv_heads = c.n_kv_heads;
  rp.n_tokens = n_tokens;
  rp.head_dim = c.head_dim;
  FCG_DEVICE(lib);
  FCG_ORDER(lib, static_cast<cudaStream_t>(stream));
  FCG_CUDA(fcg::launch_register_copy(rp, static_cast<cudaStream_t>(stream)));
  lib->stats.register_launches++;
  {
    fcg_status_t mst = mark_last(lib, static_cast<cudaStream_t>(stream));
    if (mst != FCG_OK) return mst;
  }

  commit_segment_slot(lib, sl, n_tokens, orig_start);
  *seg_id_out = sid;
  return FCG_OK;
}

// ------------------------------------------------------------------ NEXT-4: fp8 (e4m3) segment storage (R26)
fcg_status_t fcg_segment_register_fp8(fcg_library_t *lib, const void *k, const void *v, int32_t n_tokens, int32_t orig_start,
                                      const int64_t *strides, void *stream, int32_t *seg_id_out) {
  if (!lib || !k || !v || !seg_id_out) return fail(FCG_ERR_INVALID_ARG, "NULL argument");
  if (n_tokens <= 0 || orig_start < 0) return fail(FCG_ERR_INVALID_ARG, "n_tokens must be > 0 and orig_start >= 0");
  const fcg_config_t &c = lib->cfg;
  int64_t st[4] = {(int64_t)c.n_kv_heads * n_tokens * c.head_dim, (int64_t)n_tokens * c.head_dim, c.head_dim, 1};
  if (strides) {
    if (strides[3] != 1) return fail(FCG_ERR_INVALID_ARG, "strides[3] must be 1 (contiguous head_dim)");
    for (int i = 0; i < 3; ++i) {
      if (strides[i] % 8) return fail(FCG_ERR_INVALID_ARG, "strides must be multiples of 8 elements (16-byte rows)");
      st[i] = strides[i];
    }
  }
  if (((uintptr_t)k % 16) || ((uintptr_t)v % 16)) return fail(FCG_ERR_INVALID_ARG, "k and v must be 16-byte aligned");
  SegmentSlot sl;
  fcg_status_t sst = find_segment_slot(lib, n_tokens, sl, FCG_STORE_FP8_E4M3);
  if (sst != FCG_OK) return sst;
  const uint64_t codes = lib->fp8_code_bytes(n_tokens), half = sl.bytes / 2;
  fcg::RegisterFp8Params rp;
  rp.k_src = static_cast<const uint16_t *>(k);
  rp.v_src = static_cast<const uint16_t *>(v);
  rp.k_dst = lib->arena + sl.off;
  rp.k_exp = lib->arena + sl.off + codes;
  rp.v_dst = lib->arena + sl.off + half;
  rp.v_exp = lib->arena + sl.off + half + codes;
  rp.s_layer = st[0];
  rp.s_head = st[1];
  rp.s_tok = st[2];
  rp.n_layers = c.n_layers;
  rp.n_kv_heads = c.n_kv_heads;
  rp.n_tokens = n_tokens;
  rp.head_dim = c.head_dim;
  FCG_DEVICE(lib);
  FCG_ORDER(lib, static_cast<cudaStream_t>(stream));
  FCG_CUDA(fcg::launch_register_fp8(rp, static_cast<cudaStream_t>(stream)));
  lib->stats.register_launches++;
  {
    fcg_status_t mst = mark_last(lib, static_cast<cudaStream_t>(stream));
    if (mst != FCG_OK) return mst;
  }
  commit_segment_slot(lib, sl, n_tokens, orig_start, FCG_STORE_FP8_E4M3);
  *seg_id_out = sl.sid;
  return FCG_OK;
}

fcg_status_t fcg_segment_storage(fcg_library_t *lib, int32_t seg_id, int32_t *format, uint64_t *bytes) {
  if (!lib) return fail(FCG_ERR_INVALID_ARG, "lib is NULL");
  if (seg_id < 0 || seg_id >= lib->cfg.max_segments || !lib->segments[seg_id].live)
    return fail(FCG_ERR_BAD_SEGMENT, "unknown segment %d", seg_id);
  if (format) *format = lib->segments[seg_id].fmt;
  if (bytes) *bytes = lib->segments[seg_id].bytes;
  return FCG_OK;
}

fcg_status_t fcg_segment_read(fcg_library_t *lib, int32_t seg_id, void *k_out, void *v_out, void *k_exp_out, void *v_exp_out,
                              void *stream_) {
  if (!lib || !k_out || !v_out) return fail(FCG_ERR_INVALID_ARG, "NULL argument");
  if (seg_id < 0 || seg_id >= lib->cfg.max_segments || !lib->segments[seg_id].live)
    return fail(FCG_ERR_BAD_SEGMENT, "unknown segment %d", seg_id);
  const SegmentRec &s = lib->segments[seg_id];
  const fcg_config_t &c = lib->cfg;
  cudaStream_t stream = static_cast<cudaStream_t>(stream_);
  const unsigned char *base = (s.resident ? lib->arena : lib->host_arena) + s.offset;
  const uint64_t rows = (uint64_t)c.n_layers * c.n_kv_heads * (uint64_t)s.n_tokens;
  const bool fp8 = s.fmt == FCG_STORE_FP8_E4M3;
  if (fp8 && (!k_exp_out || !v_exp_out)) return fail(FCG_ERR_INVALID_ARG, "an fp8 segment needs k_exp_out and v_exp_out");
  const uint64_t payload = rows * (fp8 ? (uint64_t)c.head_dim : lib->kv_row_bytes());
  FCG_DEVICE(lib);
  FCG_ORDER(lib, stream);
  FCG_CUDA(cudaMemcpyAsync(k_out, base, payload, cudaMemcpyDefault, stream));
  FCG_CUDA(cudaMemcpyAsync(v_out, base + s.bytes / 2, payload, cudaMemcpyDefault, stream));
  if (fp8) {
    const uint64_t codes = lib->fp8_code_bytes(s.n_tokens);
    FCG_CUDA(cudaMemcpyAsync(k_exp_out, base + codes, rows, cudaMemcpyDefault, stream));
    FCG_CUDA(cudaMemcpyAsync(v_exp_out, base + s.bytes / 2 + codes, rows, cudaMemcpyDefault, stream));
  }
  return mark_last(lib, stream);
}

// ------------------------------------------------------------------ NEXT-3: two-tier residency
fcg_status_t fcg_segment_offload(fcg_library_t *lib, int32_t seg_id, void *stream) {
  if (!lib) return fail(FCG_ERR_INVALID_ARG, "lib is NULL");
  if (seg_id < 0 || seg_id >= lib->cfg.max_segments || !lib->segments[seg_id].live)
    return fail(FCG_ERR_BAD_SEGMENT, "unknown segment %d", seg_id);
  if (!lib->host_arena) return fail(FCG_ERR_INVALID_ARG, "the library was created without a host tier (host_arena)");
  SegmentRec &s = lib->segments[seg_id];
  if (!s.resident) return FCG_OK;
  const size_t fi = range_find(lib->host_free, s.bytes);
  if (fi == lib->host_free.size())
    return fail(FCG_ERR_OUT_OF_ARENA, "no free host-tier range of %llu bytes for segment %d", (unsigned long long)s.bytes, seg_id);
  const uint64_t hoff = lib->host_free[fi].off;
  FCG_DEVICE(lib);
  FCG_ORDER(lib, static_cast<cudaStream_t>(stream));
  FCG_CUDA(cudaMemcpyAsync(lib->host_arena + hoff, lib->arena + s.offset, s.bytes, cudaMemcpyDeviceToHost,
                           static_cast<cudaStream_t>(stream)));
  {
    fcg_status_t mst = mark_last(lib, static_cast<cudaStream_t>(stream));
    if (mst != FCG_OK) return mst;
  }
  range_take(lib->host_free, fi, s.bytes);
  range_give(lib->seg_free, s.offset, s.bytes);
  s.offset = hoff;
  s.resident = false;
  lib->stats.offload_copies++;
  return FCG_OK;
}

fcg_status_t fcg_segment_prefetch(fcg_library_t *lib, int32_t seg_id, void *stream) {
  if (!lib) return fail(FCG_ERR_INVALID_ARG, "lib is NULL");
  if (seg_id < 0 || seg_id >= lib->cfg.max_segments || !lib->segments[seg_id].live)
    return fail(FCG_ERR_BAD_SEGMENT, "unknown segment %d", seg_id);
  if (!lib->host_arena) return fail(FCG_ERR_INVALID_ARG, "the library was created without a host tier (host_arena)");
  SegmentRec &s = lib->segments[seg_id];
  if (s.resident) return FCG_OK;
  const size_t fi = range_find(lib->seg_free, s.bytes);
  if (fi == lib->seg_free.size())
    return fail(FCG_ERR_OUT_OF_ARENA, "no free arena range of %llu bytes for segment %d", (unsigned long long)s.bytes, seg_id);
  const uint64_t off = lib->seg_free[fi].off;
  FCG_DEVICE(lib);
  FCG_ORDER(lib, static_cast<cudaStream_t>(stream));
  FCG_CUDA(cudaMemcpyAsync(lib->arena + off, lib->host_arena + s.offset, s.bytes, cudaMemcpyHostToDevice,
                           static_cast<cudaStream_t>(stream)));
  {
    fcg_status_t mst = mark_last(lib, static_cast<cudaStream_t>(stream));
    if (mst != FCG_OK) return mst;
  }
  range_take(lib->seg_free, fi, s.bytes);
  range_give(lib->host_free, s.offset, s.bytes);
  s.offset = off;
  s.resident = true;
  lib->stats.prefetch_copies++;
  return FCG_OK;
}

fcg_status_t fcg_segment_info(fcg_library_t *lib, int32_t seg_id, int32_t *n_tokens, int32_t *orig_start, int32_t *resident) {
  if (!lib) return fail(FCG_ERR_INVALID_ARG, "lib is NULL");
  if (seg_id < 0 || seg_id >= lib->cfg.max_segments || !lib->segments[seg_id].live)
    return fail(FCG_ERR_BAD_SEGMENT, "unknown segment %d", seg_id);
  const SegmentRec &s = lib->segments[seg_id];
  if (n_tokens) *n_tokens = s.n_tokens;
  if (orig_start) *orig_start = s.orig_start;
  if (resident) *resident = s.resident ? 1 : 0;
  return FCG_OK;
}

fcg_status_t fcg_segment_release(fcg_library_t *lib, int32_t seg_id) {
  if (!lib) return fail(FCG_ERR_INVALID_ARG, "lib is NULL");
  if (seg_id < 0 || seg_id >= lib->cfg.max_segments || !lib->segments[seg_id].live)
    return fail(FCG_ERR_BAD_SEGMENT, "unknown segment %d", seg_id);
  SegmentRec &s = lib->segments[seg_id];
  range_give(s.resident ? lib->seg_free : lib->host_free, s.offset, s.bytes);
  s.live = false;
  s.resident = true;
  lib->n_segments_live--;
  return FCG_OK;
}

// ------------------------------------------------------------------------------------- S2 + S3
namespace {
struct CheckedPlan {
  int32_t capacity, T, n_pages;
  std::vector<int32_t> deltas;
};

fcg_status_t validate_plan(fcg_library *lib, const fcg_plan_t &pl, CheckedPlan &cp) {
  const fcg_config_t &c = lib->cfg;
  if (pl.task_id < 0 || pl.task_id >= c.max_tasks) return fail(FCG_ERR_BAD_TASK, "task id %d out of range", pl.task_id);
  if (lib->tasks[pl.task_id].live) return fail(FCG_ERR_BAD_TASK, "task %d is already live", pl.task_id);
  if (pl.n_entries < 0 || pl.n_holes < 0 || (pl.n_entries > 0 && !pl.entries) || (pl.n_holes > 0 && !pl.holes))
    return fail(FCG_ERR_INVALID_ARG, "plan arrays");
  if (pl.n_entries + pl.n_holes == 0) return fail(FCG_ERR_INVALID_ARG, "empty plan");
  std::vector<std::pair<int64_t, int64_t>> spans;
  spans.reserve(pl.n_entries + pl.n_holes);
  cp.deltas.clear();
  for (int i = 0; i < pl.n_entries; ++i) {
    const fcg_plan_entry_t &e = pl.entries[i];
    if (e.seg_id < 0 || e.seg_id >= c.max_segments || !lib->segments[e.seg_id].live)
      return fail(FCG_ERR_BAD_SEGMENT, "entry %d: unknown segment %d", i, e.seg_id);
    const SegmentRec &s = lib->segments[e.seg_id];
    if (e.n_tokens <= 0 || e.src_begin < 0 || (int64_t)e.src_begin + e.n_tokens > s.n_tokens || e.dst_offset < 0)
      return fail(FCG_ERR_RANGE, "entry %d: source/destination range", i);
    spans.push_back({e.dst_offset, (int64_t)e.dst_offset + e.n_tokens});
    cp.deltas.push_back(e.dst_offset - s.orig_start - e.src_begin);
  }
  for (int i = 0; i < pl.n_holes; ++i) {
    const fcg_hole_t &h = pl.holes[i];
    if (h.n_tokens <= 0 || h.begin < 0) return fail(FCG_ERR_RANGE, "hole %d: range", i);
    spans.push_back({h.begin, (int64_t)h.begin + h.n_tokens});
  }
  int64_t T = 0;
  for (auto &s : spans) T = std::max(T, s.second);
  const int64_t cap = pl.capacity_tokens > 0 ? pl.capacity_tokens : T;
  if (T > cap) return fail(FCG_ERR_RANGE, "plan ends at %lld, beyond capacity_tokens %lld", (long long)T, (long long)cap);
  if (cap > c.max_task_tokens) return fail(FCG_ERR_RANGE, "capacity %lld exceeds max_task_tokens %d", (long long)cap, c.max_task_tokens);
  std::sort(spans.begin(), spans.end());
  for (size_t i = 1; i < spans.size(); ++i)
    if (spans[i].first < spans[i - 1].second) return fail(FCG_ERR_OVERLAP, "entries/holes overlap at token %lld", (long long)spans[i].first);
  cp.capacity = (int32_t)cap;
  cp.T = (int32_t)T;
  cp.n_pages = (int32_t)((cap + c.page_size - 1) / c.page_size);
  return FCG_OK;
}
}  // namespace

}  // extern "C"

namespace {
// fcg_stitch / fcg_stitch_prefetch.  `prefetch`: offloaded segments named by the plans are first copied back to the
// device tier on the library's copy stream (first-fit arena range; a segment that finds no room stays where it is and
// is read in place) while the entries of the resident segments are stitched on `stream`; the entries of the prefetched
// segments follow in a second launch once the copies have landed.  Page allocation does not depend on the mode.
fcg_status_t stitch_impl(fcg_library *lib, const fcg_plan_t *plans, int32_t n_plans, cudaStream_t stream, bool prefetch) {
  const fcg_config_t &c = lib->cfg;
  std::vector<CheckedPlan> checked(n_plans);
  int64_t need_pages = 0;
  for (int i = 0; i < n_plans; ++i) {
    for (int j = 0; j < i; ++j)
      if (plans[j].task_id == plans[i].task_id) return fail(FCG_ERR_BAD_TASK, "task id %d repeated in the batch", plans[i].task_id);
    fcg_status_t st = validate_plan(lib, plans[i], checked[i]);
    if (st != FCG_OK) return st;
    need_pages += checked[i].n_pages;
  }
  if (need_pages > (int64_t)lib->page_stack.size())
    return fail(FCG_ERR_OUT_OF_PAGES, "need %lld pages, %zu free", (long long)need_pages, lib->page_stack.size());

  // ---- prefetch planning: arena ranges for the offloaded segments the plans name (nothing committed yet) ----
  struct Move {
    int32_t seg;
    uint64_t dev_off, host_off, bytes;
  };
  std::vector<Move> moves;
  std::vector<FreeRange> seg_free = lib->seg_free;              // a copy: committed at the end
  if (prefetch && lib->host_arena) {
    for (int i = 0; i < n_plans; ++i)
      for (int e = 0; e < plans[i].n_entries; ++e) {
        const int32_t sid = plans[i].entries[e].seg_id;
        const SegmentRec &s = lib->segments[sid];
        if (s.resident) continue;
        bool seen = false;
        for (auto &m : moves) seen |= m.seg == sid;
        if (seen) continue;
        const size_t fi = range_find(seg_free, s.bytes);
        if (fi == seg_free.size()) continue;                      // no room: this one is read in place
        moves.push_back({sid, seg_free[fi].off, s.offset, s.bytes});
        range_take(seg_free, fi, s.bytes);
      }
  }
  auto move_of = [&](int32_t sid) -> const Move * {
    for (auto &m : moves)
      if (m.seg == sid) return &m;
    return nullptr;
  };

  // ---- build the launches (host): gb = entries of resident (or in-place) segments + all page ids, gb2 = entries of
  // the segments being prefetched ----------------------------------------------------------------------------------
  const int P = c.page_size;
  GatherBuilder gb, gb2;
  // page ids are taken from a COPY of the stack; committed only when everything has been enqueued
  std::vector<int32_t> stack = lib->page_stack;
  std::vector<int64_t> plan_page_base(n_plans);
  for (int i = 0; i < n_plans; ++i) {
    plan_page_base[i] = (int64_t)gb.pages.size();
    for (int k = 0; k < checked[i].n_pages; ++k) {
      gb.pages.push_back(stack.back());
      stack.pop_back();
    }
    for (int e = 0; e < plans[i].n_entries; ++e) {
      const fcg_plan_entry_t &pe = plans[i].entries[e];
      const SegmentRec &s = lib->segments[pe.seg_id];
      const Move *mv = move_of(pe.seg_id);
      GatherBuilder &g = mv ? gb2 : gb;
      fcg::StitchEntryDev de;
      // an offloaded segment is read in place from the pinned host tier (or from the arena range it is being
      // prefetched into); an fp8 segment is de-quantised on the way
      if (mv) {
        SegmentRec moved = s;
        moved.offset = mv->dev_off;
        moved.resident = true;
        g.source_segment(lib, moved, de);
      } else {
        g.source_segment(lib, s, de);
      }
      g.pool_side(lib, de.k_dst, de.v_dst, de.dst_layer_stride, de.dst_head_stride);
      de.table_off = g.table_for(lib, checked[i].deltas[e]);
      const int32_t ei = (int32_t)g.entries.size();
      g.entries.push_back(de);
      // chunks: one per destination page touched
      int32_t done = 0;
      while (done < pe.n_tokens) {
        const int32_t dst = pe.dst_offset + done;
        const int32_t slot0 = dst % P;
        const int32_t n = std::min(P - slot0, pe.n_tokens - done);
        fcg::StitchChunkDev dc;
        dc.entry = ei;
        dc.dst_tok = g.pool_tok(lib, gb.pages[plan_page_base[i] + dst / P], slot0);
        dc.src_tok = pe.src_begin + done;
        dc.ntok = n;
        g.chunks.push_back(dc);
        done += n;
      }
    }
  }

  // ---- the last host-side checks, BEFORE anything is enqueued (fcg.h conventions; enqueue_gather repeats them) -----
  if (gb.blob_bytes() > BLOB_BYTES || gb2.blob_bytes() > BLOB_BYTES)
    return fail(FCG_ERR_OUT_OF_ARENA, "plan blob of %llu bytes exceeds %llu (fewer entries / plans per call)",
                (unsigned long long)std::max(gb.blob_bytes(), gb2.blob_bytes()), (unsigned long long)BLOB_BYTES);
  if ((uint64_t)c.n_pages * c.n_kv_heads * c.page_size > 0x7fffffffull) return fail(FCG_ERR_INVALID_ARG, "pool too large for 32-bit row offsets");

  // ---- enqueue: copies, blob, kernel, page tables -----------------------------------------------
  FCG_DEVICE(lib);
  FCG_ORDER(lib, stream);
  if (!moves.empty()) {
    // the copy stream starts after whatever used the library last (the arena ranges it writes may have just been freed)
    if (lib->have_last) FCG_CUDA(cudaStreamWaitEvent(lib->copy_stream, lib->last_ev, 0));
    for (auto &m : moves)
      FCG_CUDA(cudaMemcpyAsync(lib->arena + m.dev_off, lib->host_arena + m.host_off, m.bytes, cudaMemcpyHostToDevice, lib->copy_stream));
    FCG_CUDA(cudaEventRecord(lib->prefetch_ev, lib->copy_stream));
  }
  GatherBlob gbl;
  fcg_status_t st = enqueue_gather(lib, gb, stream, gbl);
  if (st != FCG_OK) return st;
  for (int i = 0; i < n_plans; ++i) {
    int32_t *dst = lib->tables() + (int64_t)plans[i].task_id * lib->pages_per_task;
    FCG_CUDA(cudaMemcpyAsync(dst, gbl.slot->dev + gbl.off_pages + plan_page_base[i] * sizeof(int32_t),
                             (size_t)checked[i].n_pages * sizeof(int32_t), cudaMemcpyDeviceToDevice, stream));
  }
  GatherBlob gbl2;
  if (!moves.empty()) {
    FCG_CUDA(cudaStreamWaitEvent(stream, lib->prefetch_ev, 0));
    st = enqueue_gather(lib, gb2, stream, gbl2);
    if (st != FCG_OK) return st;
  }
  st = mark_last(lib, stream);
  if (st != FCG_OK) return st;
  const int32_t *pages = gb.pages.data();

  // ---- commit ------------------------------------------------------------------------------------
  lib->page_stack.swap(stack);
  if (!moves.empty()) {
    lib->seg_free.swap(seg_free);
    for (auto &m : moves) {
      SegmentRec &s = lib->segments[m.seg];
      range_give(lib->host_free, m.host_off, m.bytes);
      s.offset = m.dev_off;
      s.resident = true;
      lib->stats.prefetch_copies++;
    }
  }
  for (int i = 0; i < n_plans; ++i) {
    TaskRec &t = lib->tasks[plans[i].task_id];
    t.live = true;
    t.gen = ++lib->task_gen;
    t.capacity = checked[i].capacity;
    t.n_tokens = checked[i].T;
    t.pages.assign(pages + plan_page_base[i], pages + plan_page_base[i] + checked[i].n_pages);
    t.filled.assign(t.capacity, 0);
    t.spans.clear();
    for (int e = 0; e < plans[i].n_entries; ++e) {
      const fcg_plan_entry_t &pe = plans[i].entries[e];
      std::fill(t.filled.begin() + pe.dst_offset, t.filled.begin() + pe.dst_offset + pe.n_tokens, (uint8_t)1);
      t.spans.push_back({pe.dst_offset, pe.n_tokens});
    }
    t.filled_prefix = 0;
    while (t.filled_prefix < t.capacity && t.filled[t.filled_prefix]) t.filled_prefix++;
    lib->n_tasks_live++;
  }
  return FCG_OK;
}
}  // namespace

extern "C" {

fcg_status_t fcg_stitch(fcg_library_t *lib, const fcg_plan_t *plans, int32_t n_plans, void *stream) {
  if (!lib || !plans || n_plans <= 0) return fail(FCG_ERR_INVALID_ARG, "NULL / empty plan array");
  return stitch_impl(lib, plans, n_plans, static_cast<cudaStream_t>(stream), false);
}

fcg_status_t fcg_stitch_prefetch(fcg_library_t *lib, const fcg_plan_t *plans, int32_t n_plans, void *stream) {
  if (!lib || !plans || n_plans <= 0) return fail(FCG_ERR_INVALID_ARG, "NULL / empty plan array");
  return stitch_impl(lib, plans, n_plans, static_cast<cudaStream_t>(stream), true);
}

// ------------------------------------------------------------------------------------ S4 + S5/S6
namespace {

// choose the number of KV splits for `base` CTAs per split so that waves on the GPU are well filled
// without paying much for fp32 partials.
int choose_splits(int64_t base_ctas, int tiles, int rows, int head_dim, int ctas_per_sm, int n_sms) {
  if (tiles <= 1) return 1;
  const double slots = (double)n_sms * ctas_per_sm;
  // everything in bytes streamed by one SM (an SM's share of HBM is ~44 GB/s: 10 us ~ 440 KB)
  // launch + prologue + epilogue of a CTA.  head_dim 256: a 64 KB Q tile to fill and a 5-stage ring to ramp -- measured on
  // the 4k-token decode step (336 CTAs unsplit: 0.26 ms; 4 / 8 / 16 splits: 0.29 / 0.34 / 0.50 ms), ~6 us per extra CTA
  const double kFixedPerCta = head_dim > 128 ? 250000.0 : 6000.0;
  const double kCombineLaunch = 400000.0;        // the extra combine kernel: launch gap + its own ramp
  double best_cost = 1e30, cost_1 = 1e30;
  int best = 1;
  const int max_s = std::min(tiles, 64);
  for (int s = 1; s <= max_s; ++s) {
    const int tiles_per = (tiles + s - 1) / s;
    const int s_eff = (tiles + tiles_per - 1) / tiles_per;
    if (s_eff != s) continue;
    // every (row group, split) CTA counts, also those of a row group that stops early (a hole in the middle of the cache):
    // counting only the non-empty ones picked 12 splits instead of 9 for one layer of C3 and took 51 us instead of 37
    const double ctas = (double)base_ctas * s;
    const double waves = ceil(ctas / slots);
    // time ~ waves * (one CTA's K/V stream + its fp32 partial rows), plus what the combine kernel reads and writes
    const double kv_bytes = (double)tiles_per * KV_TILE * head_dim * 4.0;
    const double part_bytes = s > 1 ? (double)rows * (head_dim + 2) * 4.0 : 0.0;
    const double combine = s > 1 ? kCombineLaunch + ctas * part_bytes / n_sms : 0.0;
    const double cost = waves * (kv_bytes + part_bytes + kFixedPerCta) + combine;
    if (s == 1) cost_1 = cost;
    if (cost < best_cost * 0.999) {
      best_cost = cost;
      best = s;
    }
  }
  // a split must pay for itself with margin: partials are fp32 and the measured cost of splitting when the grid
  // already fills the GPU is 20-25 % (C3: 0.41 ms unsplit, 0.50 ms with two splits)
  return best_cost < 0.85 * cost_1 ? best : 1;
}

// What a patch is, independent of the tensors it is run on: the tasks, their position lists and the layer count per call.
struct PatchSpec {
  const int32_t *task_ids;
  const int32_t *n_per_task;
  int32_t n_tasks;
  const int32_t *positions;
  int32_t n_layers;           // layers per call (split selection, partial sizing)
};

// the tensors and the layer range of one call
struct PatchIO {
  int32_t layer_begin, n_layers;
  const void *q, *k, *v;
  void *out;
  cudaStream_t stream;
};

struct PatchCheck {
  int64_t n_total = 0;
  std::vector<int32_t> new_capacity;   // per task: capacity after this patch (R25: appends grow the task)
  std::vector<int32_t> new_pages;      // per task: pages to add
  int64_t pages_needed = 0;
};

// Host-side validation of a patch; touches nothing (fcg.h conventions: a failing call leaves the library unchanged and
// launches nothing).  R6: every position a query sees is filled by earlier work or by this call.  R25: positions at or
// beyond the capacity append -- the task grows to positions[n-1] + 1 <= max_task_tokens, pages come on demand.
fcg_status_t validate_patch(fcg_library *lib, const PatchSpec &ps, PatchCheck &ck) {
  const fcg_config_t &c = lib->cfg;
  if (!ps.positions || !ps.task_ids || !ps.n_per_task || ps.n_tasks <= 0) return fail(FCG_ERR_INVALID_ARG, "NULL / empty argument");
  // the attention grids run (layer, task) along z and kv heads along y: CUDA's limit for both is 65535
  if ((int64_t)ps.n_layers * ps.n_tasks > 65535 || c.n_kv_heads > 65535)
    return fail(FCG_ERR_INVALID_ARG, "%d layers x %d tasks in one call exceed the launch limit of 65535: patch fewer layers or tasks per call",
                ps.n_layers, ps.n_tasks);
  ck.n_total = 0;
  ck.pages_needed = 0;
  ck.new_capacity.assign(ps.n_tasks, 0);
  ck.new_pages.assign(ps.n_tasks, 0);
  const int P = c.page_size;
  for (int t = 0; t < ps.n_tasks; ++t) {
    const int32_t id = ps.task_ids[t];
    if (id < 0 || id >= c.max_tasks || !lib->tasks[id].live) return fail(FCG_ERR_BAD_TASK, "unknown task %d", id);
    for (int u = 0; u < t; ++u)
      if (ps.task_ids[u] == id) return fail(FCG_ERR_BAD_TASK, "task %d repeated in the batch", id);
    const int32_t n = ps.n_per_task[t];
    if (n <= 0) return fail(FCG_ERR_INVALID_ARG, "task %d: n must be > 0", id);
    const int32_t *pos = ps.positions + ck.n_total;
    for (int i = 1; i < n; ++i)
      if (pos[i] <= pos[i - 1]) return fail(FCG_ERR_INVALID_ARG, "task %d: positions must be strictly increasing", id);
    const TaskRec &tr = lib->tasks[id];
    if (pos[0] < 0 || pos[n - 1] >= c.max_task_tokens)
      return fail(FCG_ERR_RANGE, "task %d: position outside [0, max_task_tokens = %d)", id, c.max_task_tokens);
    // every x <= pos[n-1] must be filled by earlier work or by this call (positions beyond the capacity are unfilled)
    int pi = 0;
    for (int32_t x = tr.filled_prefix; x <= pos[n - 1]; ++x) {
      while (pi < n && pos[pi] < x) ++pi;
      const bool was = x < tr.capacity && tr.filled[x];
      if (!was && !(pi < n && pos[pi] == x))
        return fail(FCG_ERR_UNFILLED, "task %d: position %d is visible to a patch query but was never filled", id, x);
    }
    ck.new_capacity[t] = std::max(tr.capacity, pos[n - 1] + 1);
    ck.new_pages[t] = std::max<int32_t>(0, (ck.new_capacity[t] + P - 1) / P - (int32_t)tr.pages.size());
    ck.pages_needed += ck.new_pages[t];
    ck.n_total += n;
  }
  if (ck.n_total > (1 << 20)) return fail(FCG_ERR_INVALID_ARG, "too many patch tokens in one call");
  if (ck.pages_needed > (int64_t)lib->page_stack.size())
    return fail(FCG_ERR_OUT_OF_PAGES, "need %lld pages to grow, %zu free", (long long)ck.pages_needed, lib->page_stack.size());
  return FCG_OK;
}

fcg_status_t validate_io(fcg_library *lib, const PatchIO &io) {
  const fcg_config_t &c = lib->cfg;
  if (!io.q || !io.k || !io.v || !io.out) return fail(FCG_ERR_INVALID_ARG, "NULL / empty argument");
  if (io.layer_begin < 0 || io.n_layers <= 0 || io.layer_begin + io.n_layers > c.n_layers)
    return fail(FCG_ERR_INVALID_ARG, "layer range [%d, %d) outside [0, %d)", io.layer_begin, io.layer_begin + io.n_layers, c.n_layers);
  return FCG_OK;
}

// Everything the kernels need besides the tensors, as offsets into one blob (positions, per-token table offsets and
// split counts, task descriptors in call order and grouped by CTA class, page ids of growing tasks) plus the launch
// shape.  The blob lives in a transient slot (fcg_patch) or in a plan's own device range (fcg_patch_plan_create).
struct PatchLayout {
  int64_t n_total = 0;
  int32_t n_tasks = 0;
  uint64_t off_pos = 0, off_toff = 0, off_tspl = 0, off_tasks = 0, off_tasks2 = 0, off_grow = 0, used = 0;
  bool use_tc = false;
  int max_splits = 1, max_rows = 0, rows_per_cta_split = 64, max_row_groups = 1;
  int n_cls[3] = {0, 0, 0}, cls_begin[3] = {0, 0, 0}, cls_rgs[3] = {1, 1, 1};
  uint64_t off_items = 0;     // mixed-class launch: int4 {class, task index in the class-grouped list, row group, split}
  int32_t n_items = 0;
  struct Grow {
    int32_t task_id, first_lp, count;
    int64_t index;            // first page id of this task inside the off_grow region
  };
  std::vector<Grow> grows;
  std::vector<int32_t> grow_pages;
};

// fills `host` (capacity `cap` bytes) and `lay`; page ids for growth are taken from the top of a COPY of the stack
fcg_status_t build_patch_blob(fcg_library *lib, const PatchSpec &ps, const PatchCheck &ck, unsigned char *host, uint64_t cap,
                              PatchLayout &lay) {
  const fcg_config_t &c = lib->cfg;
  const int64_t n_total = ck.n_total;
  BlobWriter bw(host, cap);
  lay.n_total = n_total;
  lay.n_tasks = ps.n_tasks;
  lay.off_pos = bw.reserve(n_total * 4);
  lay.off_toff = bw.reserve(n_total * 4);
  lay.off_tspl = bw.reserve(n_total * 4);
  lay.off_tasks = bw.reserve((uint64_t)ps.n_tasks * sizeof(fcg::AttnTaskDev));
  lay.off_tasks2 = bw.reserve((uint64_t)ps.n_tasks * sizeof(fcg::AttnTaskDev));   // tcgen05 path: tasks by Q-tile class
  lay.off_grow = bw.reserve((uint64_t)std::max<int64_t>(ck.pages_needed, 1) * 4);
  if (lay.off_pos == UINT64_MAX || lay.off_toff == UINT64_MAX || lay.off_tspl == UINT64_MAX || lay.off_tasks == UINT64_MAX ||
      lay.off_tasks2 == UINT64_MAX || lay.off_grow == UINT64_MAX)
    return fail(FCG_ERR_OUT_OF_ARENA, "patch blob exceeds %llu bytes", (unsigned long long)cap);
  auto *h_pos = reinterpret_cast<int32_t *>(host + lay.off_pos);
  auto *h_toff = reinterpret_cast<int32_t *>(host + lay.off_toff);
  auto *h_tspl = reinterpret_cast<int32_t *>(host + lay.off_tspl);
  auto *h_tasks = reinterpret_cast<fcg::AttnTaskDev *>(host + lay.off_tasks);
  auto *h_grow = reinterpret_cast<int32_t *>(host + lay.off_grow);
  memcpy(h_pos, ps.positions, (size_t)n_total * 4);
  h_grow[0] = 0;

  // R25: page ids of the growing tasks, tasks in array order, ascending logical order
  lay.grows.clear();
  lay.grow_pages.clear();
  {
    size_t top = lib->page_stack.size();
    for (int t = 0; t < ps.n_tasks; ++t) {
      if (ck.new_pages[t] == 0) continue;
      PatchLayout::Grow g{ps.task_ids[t], (int32_t)lib->tasks[ps.task_ids[t]].pages.size(), ck.new_pages[t], (int64_t)lay.grow_pages.size()};
      for (int k = 0; k < g.count; ++k) lay.grow_pages.push_back(lib->page_stack[--top]);
      lay.grows.push_back(g);
    }
    if (!lay.grow_pages.empty()) memcpy(h_grow, lay.grow_pages.data(), lay.grow_pages.size() * 4);
  }

  const int G = c.n_q_heads / c.n_kv_heads;
  int max_rows = 0;
  for (int t = 0; t < ps.n_tasks; ++t) max_rows = std::max(max_rows, ps.n_per_task[t] * G);
  lay.max_rows = max_rows;
  // head_dim above 128 has ONE CTA class on the tcgen05 path (a 128-row Q tile, more rows run as more row groups); only
  // head_dim 64 and 128 have the split-KV mma.sync kernel besides (R27)
  const bool d256 = c.head_dim > 128;
  const bool tc_only = c.head_dim != 64 && c.head_dim != 128;
  if (tc_only && !lib->have_tma) return fail(FCG_ERR_CUDA, "head_dim %d needs the tcgen05 / TMA attention path, which is unavailable on this device", c.head_dim);
  const bool use_tc = lib->have_tma && (max_rows >= lib->tc_min_rows || tc_only);
  lay.use_tc = use_tc;
  // tcgen05 path: a task with <= 128 rows per kv head runs CTAs with one 128-row Q tile (deep K/V rings: the
  // HBM-bound regime), a task with more rows CTAs with two (K/V read once per 256 rows).  A batch that mixes
  // both is launched as two grids, one per class.
  lay.rows_per_cta_split = max_rows <= 16 ? 16 : (max_rows <= 32 ? 32 : 64);
  auto rows_per_cta_of = [&](int rows) { return use_tc ? ((rows > 128 && !d256) ? 256 : 128) : lay.rows_per_cta_split; };
  const int ctas_per_sm = use_tc ? fcg::attn_tc_ctas_per_sm(c.head_dim, (max_rows > 128 && !d256) ? 2 : 1, (max_rows > 64 && max_rows <= 128 && !d256) ? 2 : 1)
                                 : fcg::attn_split_ctas_per_sm(c.head_dim);
  int max_splits = 1;
  int64_t tok_off = 0;
  for (int t = 0; t < ps.n_tasks; ++t) {
    const int32_t n = ps.n_per_task[t];
    const int32_t kv_len = ps.positions[tok_off + n - 1] + 1;
    const int tiles = (kv_len + KV_TILE - 1) / KV_TILE;
    const int rows_per_cta = rows_per_cta_of(n * G);
    const int rg = (n * G + rows_per_cta - 1) / rows_per_cta;
    const int64_t base = (int64_t)rg * c.n_kv_heads * ps.n_layers * ps.n_tasks;
    int ns = lib->force_splits > 0 ? std::min(std::min(lib->force_splits, tiles), 64)      // the combine kernel holds a split per lane, twice
                                   : choose_splits(base, tiles, std::min(n * G, rows_per_cta), c.head_dim, ctas_per_sm, lib->n_sms);
    const int tiles_per = (tiles + ns - 1) / ns;
    ns = (tiles + tiles_per - 1) / tiles_per;      // no empty trailing split
    fcg::AttnTaskDev &d = h_tasks[t];
    d.table_off = ps.task_ids[t] * lib->pages_per_task;
    d.n = n;
    d.tok_off = (int32_t)tok_off;
    d.kv_len = kv_len;
    d.n_splits = ns;
    d.split_len = tiles_per * KV_TILE;
    d.pad0 = d.pad1 = 0;
    max_splits = std::max(max_splits, ns);
    for (int i = 0; i < n; ++i) {
      h_toff[tok_off + i] = d.table_off;
      h_tspl[tok_off + i] = ns;
    }
    tok_off += n;
  }
  lay.max_splits = max_splits;
  lay.max_row_groups = (max_rows + rows_per_cta_of(max_rows) - 1) / rows_per_cta_of(max_rows);
  // tcgen05 path: the same descriptors again, grouped by CTA class (rows per kv head <= 64 | <= 128 | more)
  auto *h_tasks2 = reinterpret_cast<fcg::AttnTaskDev *>(host + lay.off_tasks2);
  // (two 128-row CTAs instead of one two-Q-tile CTA for 129..256 rows was measured slower: C4 patch 3.24 vs 3.13 ms)
  auto class_of = [&](int rows) { return (rows <= 64 || d256) ? 0 : (rows <= 128 ? 1 : 2); };
  for (int cl = 0; cl < 3; ++cl) lay.n_cls[cl] = 0, lay.cls_rgs[cl] = 1;
  for (int t = 0; t < ps.n_tasks; ++t) lay.n_cls[class_of(h_tasks[t].n * G)]++;
  lay.cls_begin[0] = 0;
  lay.cls_begin[1] = lay.n_cls[0];
  lay.cls_begin[2] = lay.n_cls[0] + lay.n_cls[1];
  {
    int fill[3] = {0, 0, 0};
    for (int t = 0; t < ps.n_tasks; ++t) {
      const int cl = class_of(h_tasks[t].n * G);
      h_tasks2[lay.cls_begin[cl] + fill[cl]++] = h_tasks[t];
      const int q_tiles = cl == 2 ? 2 : 1;
      lay.cls_rgs[cl] = std::max(lay.cls_rgs[cl], (h_tasks[t].n * G + 128 * q_tiles - 1) / (128 * q_tiles));
    }
    // longest first inside a class: the grid's z index runs over (layer, task), so every layer ends with the shortest
    // CTAs of the class and the tail of the launch is short (block dispatch is greedy in index order)
    for (int cl = 0; cl < 3; ++cl)
      std::stable_sort(h_tasks2 + lay.cls_begin[cl], h_tasks2 + lay.cls_begin[cl] + lay.n_cls[cl],
                       [](const fcg::AttnTaskDev &a, const fcg::AttnTaskDev &b) { return a.kv_len > b.kv_len; });
  }
  // Work items of a mixed-class batch (one launch for all classes, fcg_attn_tc.cu attn_tc_mixed_kernel): every (task, row
  // group, split), the classes interleaved proportionally -- item i of the n_c items of class c sits at (i + 0.5) / n_c --
  // so that HBM-bound and compute-bound CTAs are resident side by side throughout the launch.
  lay.n_items = 0;
  lay.off_items = 0;
  const int n_classes = (lay.n_cls[0] > 0) + (lay.n_cls[1] > 0) + (lay.n_cls[2] > 0);
  if (use_tc && c.head_dim == 128 && n_classes >= 2 && !lib->use_pairs && lib->mix_classes) {
    struct Item {
      double key;
      int32_t cls, task, rg, split;
    };
    std::vector<Item> items;
    for (int cl = 0; cl < 3; ++cl) {
      std::vector<Item> mine;
      for (int t = 0; t < lay.n_cls[cl]; ++t) {
        const fcg::AttnTaskDev &d = h_tasks2[lay.cls_begin[cl] + t];
        const int rows_per_cta = cl == 2 ? 256 : 128;
        const int rgs = (d.n * G + rows_per_cta - 1) / rows_per_cta;
        for (int rg = 0; rg < rgs; ++rg)
          for (int sp = 0; sp < d.n_splits; ++sp) mine.push_back({0.0, cl, lay.cls_begin[cl] + t, rg, sp});
      }
      for (size_t i = 0; i < mine.size(); ++i) {
        mine[i].key = ((double)i + 0.5) / (double)mine.size();
        items.push_back(mine[i]);
      }
    }
    std::stable_sort(items.begin(), items.end(), [](const Item &a, const Item &b) { return a.key < b.key; });
    lay.off_items = bw.reserve(items.size() * 16);
    if (lay.off_items == UINT64_MAX) return fail(FCG_ERR_OUT_OF_ARENA, "patch blob exceeds %llu bytes", (unsigned long long)cap);
    auto *h_items = reinterpret_cast<int32_t *>(host + lay.off_items);
    for (size_t i = 0; i < items.size(); ++i) {
      h_items[4 * i + 0] = items[i].cls;
      h_items[4 * i + 1] = items[i].task;
      h_items[4 * i + 2] = items[i].rg;
      h_items[4 * i + 3] = items[i].split;
    }
    lay.n_items = (int32_t)items.size();
  }
  lay.used = bw.used;
  return FCG_OK;
}

// bytes of split-KV partials one call of `n_layers` layers needs
void partial_bytes(const fcg_library *lib, const PatchLayout &lay, int n_layers, uint64_t &part_o_bytes, uint64_t &part_ml_bytes) {
  const fcg_config_t &c = lib->cfg;
  const uint64_t part_rows = (uint64_t)n_layers * lay.max_splits * lay.n_total * c.n_q_heads;
  part_o_bytes = lay.max_splits > 1 ? align_up(part_rows * c.head_dim * 4) : 0;
  part_ml_bytes = lay.max_splits > 1 ? align_up(part_rows * 2 * 4) : 0;
}

// R25: page ids of the growing tasks -> their device page tables (before the scatter reads them)
fcg_status_t enqueue_growth(fcg_library *lib, const PatchLayout &lay, const unsigned char *dev_blob, cudaStream_t stream) {
  for (const auto &g : lay.grows)
    FCG_CUDA(cudaMemcpyAsync(lib->tables() + (int64_t)g.task_id * lib->pages_per_task + g.first_lp,
                             dev_blob + lay.off_grow + (uint64_t)g.index * 4, (size_t)g.count * 4, cudaMemcpyDeviceToDevice, stream));
  return FCG_OK;
}

// scatter -> attention (-> combine): kernel launches only.  `layer_slots`: the split-KV partials of layer l live in a slot
// of their own (planned calls: calls for different layers may then run concurrently, e.g. on the forked streams of a
// captured graph); otherwise they sit at the start of the scratch area (calls are ordered by R29).
fcg_status_t launch_patch(fcg_library *lib, const PatchLayout &lay, const unsigned char *dev_blob, const PatchIO &io, bool layer_slots = false) {
  const fcg_config_t &c = lib->cfg;
  uint64_t part_o_bytes, part_ml_bytes;
  partial_bytes(lib, lay, io.n_layers, part_o_bytes, part_ml_bytes);
  uint64_t part_o_off = 0, part_ml_off = part_o_bytes;
  if (layer_slots && lay.max_splits > 1) {
    uint64_t o1, ml1, o_all, ml_all;
    partial_bytes(lib, lay, 1, o1, ml1);
    partial_bytes(lib, lay, c.n_layers, o_all, ml_all);
    // two arrays indexed by the absolute layer: [n_layers][splits][rows][D] and [n_layers][splits][rows][2]
    const uint64_t rows1 = (uint64_t)lay.max_splits * lay.n_total * c.n_q_heads;
    part_o_off = (uint64_t)io.layer_begin * rows1 * c.head_dim * 4;
    part_ml_off = o_all + (uint64_t)io.layer_begin * rows1 * 2 * 4;
    part_o_bytes = o_all;
    part_ml_bytes = ml_all;
  }
  if (part_o_bytes + part_ml_bytes > lib->scratch_bytes)
    return fail(FCG_ERR_OUT_OF_ARENA, "workspace too small for %d-way split partials (%llu bytes)", lay.max_splits,
                (unsigned long long)(part_o_bytes + part_ml_bytes));
  const int G = c.n_q_heads / c.n_kv_heads;
  fcg::ScatterParams sp;
  sp.k_new = static_cast<const uint16_t *>(io.k);
  sp.v_new = static_cast<const uint16_t *>(io.v);
  sp.k_pool = lib->k_pool();
  sp.v_pool = lib->v_pool();
  sp.tables = lib->tables();
  sp.positions = reinterpret_cast<const int32_t *>(dev_blob + lay.off_pos);
  sp.tok_table_off = reinterpret_cast<const int32_t *>(dev_blob + lay.off_toff);
  sp.n_layers = io.n_layers;
  sp.layer_begin = io.layer_begin;
  sp.n_total = (int32_t)lay.n_total;
  sp.n_kv_heads = c.n_kv_heads;
  sp.head_dim = c.head_dim;
  sp.page_size = c.page_size;
  sp.n_pages = c.n_pages;
  FCG_CUDA(fcg::launch_scatter(sp, io.stream));
  lib->stats.scatter_launches++;

  fcg::AttnParams ap;
  ap.q = static_cast<const uint16_t *>(io.q);
  ap.out = static_cast<uint16_t *>(io.out);
  ap.k_pool = lib->k_pool();
  ap.v_pool = lib->v_pool();
  ap.tables = lib->tables();
  ap.positions = sp.positions;
  ap.tasks = reinterpret_cast<const fcg::AttnTaskDev *>(dev_blob + lay.off_tasks);
  ap.tok_splits = reinterpret_cast<const int32_t *>(dev_blob + lay.off_tspl);
  ap.part_o = reinterpret_cast<float *>(lib->arena + lib->scratch_off + part_o_off);
  ap.part_ml = reinterpret_cast<float *>(lib->arena + lib->scratch_off + part_ml_off);
  ap.n_total = (int32_t)lay.n_total;
  ap.n_layers = io.n_layers;
  ap.layer_begin = io.layer_begin;
  ap.n_q_heads = c.n_q_heads;
  ap.n_kv_heads = c.n_kv_heads;
  ap.group = G;
  ap.page_size = c.page_size;
  ap.n_tasks = lay.n_tasks;
  ap.max_splits = lay.max_splits;
  ap.max_row_groups = lay.max_row_groups;
  ap.n_pages = c.n_pages;
  ap.scale_log2 = (float)(1.4426950408889634 / sqrt((double)c.head_dim));
  ap.items = nullptr;
  ap.n_items = 0;
  ap.head_dim = c.head_dim;
  if (lay.use_tc && lay.n_items > 0) {
    // all classes in one launch, interleaved (see build_patch_blob)
    fcg::AttnParams apm = ap;
    apm.tasks = reinterpret_cast<const fcg::AttnTaskDev *>(dev_blob + lay.off_tasks2);
    apm.items = reinterpret_cast<const int4 *>(dev_blob + lay.off_items);
    apm.n_items = lay.n_items;
    FCG_CUDA(fcg::launch_attn_tc_mixed(apm, &lib->tm_k, &lib->tm_v, io.stream));
    lib->stats.attn_tc_launches++;
    lib->stats.last_attn_path = 2;
  } else if (lay.use_tc) {
    // class 0: rows replicated 2x / 4x in one softmax warpgroup (HBM-bound; the deep K/V rings matter most);
    // class 1: two tile-parity softmax warpgroups; class 2: two Q tiles per CTA
    // launched longest-CTA class first, so that the tail of the batch is made of the short CTAs
    for (int cl = 2; cl >= 0; --cl) {
      if (lay.n_cls[cl] == 0) continue;
      const int q_tiles = cl == 2 ? 2 : 1, parity_streams = cl == 1 ? 2 : 1;
      fcg::AttnParams apc = ap;
      apc.tasks = reinterpret_cast<const fcg::AttnTaskDev *>(dev_blob + lay.off_tasks2) + lay.cls_begin[cl];
      apc.n_tasks = lay.n_cls[cl];
      apc.max_row_groups = lay.cls_rgs[cl];
      if (cl == 2 && c.head_dim == 128 && lib->use_pairs)
        FCG_CUDA(fcg::launch_attn_pair(apc, &lib->tm_k, &lib->tm_v, io.stream));
      else
        FCG_CUDA(fcg::launch_attn_tc(apc, c.head_dim, q_tiles, parity_streams, &lib->tm_k, &lib->tm_v, io.stream));
      lib->stats.attn_tc_launches++;
    }
    lib->stats.last_attn_path = 2;
  } else {
    FCG_CUDA(fcg::launch_attn_split(ap, c.head_dim, lay.rows_per_cta_split, io.stream));
    lib->stats.attn_split_launches++;
    lib->stats.last_attn_path = 1;
  }
  lib->stats.last_attn_splits = lay.max_splits;
  if (lay.max_splits > 1) {
    FCG_CUDA(fcg::launch_attn_combine(ap, c.head_dim, io.stream));
    lib->stats.attn_combine_launches++;
    // The host variants stage q / k / v in the last <= scratch_total / 2 bytes of the scratch area from the copy stream,
    // which is ordered after staging_ev only (not after `stream`).  Partials that reach into the upper half may lie where
    // the next host call stages: they count as a use of the staging area until the combine kernel has read them.
    // (Planned calls keep their per-layer slots inside the lower half: fcg_patch_plan_create.)
    if (!layer_slots && part_ml_off + part_ml_bytes > lib->scratch_total / 2) {
      FCG_CUDA(cudaEventRecord(lib->staging_ev, io.stream));
      lib->have_staging_ev = true;
    }
  }
  return FCG_OK;
}

// fill state, capacity and page tables of the patched tasks (after everything has been enqueued)
void commit_patch(fcg_library *lib, const PatchSpec &ps, const PatchCheck &ck, const PatchLayout &lay) {
  for (const auto &g : lay.grows) {
    TaskRec &tr = lib->tasks[g.task_id];
    for (int k = 0; k < g.count; ++k) {
      tr.pages.push_back(lay.grow_pages[g.index + k]);
      lib->page_stack.pop_back();
    }
  }
  int64_t tok_off = 0;
  for (int t = 0; t < ps.n_tasks; ++t) {
    TaskRec &tr = lib->tasks[ps.task_ids[t]];
    const int32_t n = ps.n_per_task[t];
    if (ck.new_capacity[t] > tr.capacity) {
      tr.capacity = ck.new_capacity[t];
      tr.filled.resize(tr.capacity, 0);
    }
    for (int i = 0; i < n; ++i) tr.filled[ps.positions[tok_off + i]] = 1;
    while (tr.filled_prefix < tr.capacity && tr.filled[tr.filled_prefix]) tr.filled_prefix++;
    tr.n_tokens = std::max(tr.n_tokens, ps.positions[tok_off + n - 1] + 1);
    tok_off += n;
  }
}

// Upload the plan blob of a patch NOW and leave it in the reuse cache.  The host variants call this before they enqueue
// their big host->device copies: the blob upload of the first layer group is a small H2D copy, and the copy engine
// serves copies in issue order -- queued behind hundreds of MB of q / k / v it held back the first group's kernels until
// every byte of the call had arrived (C4: the pipelined host call took 11.1 ms, as long as copies and kernels back to
// back).  Changes no library state; the patch_common calls that follow find the same bytes cached.
fcg_status_t prime_patch_blob(fcg_library *lib, const PatchSpec &ps, const PatchCheck &ck, cudaStream_t stream, cudaStream_t consumer) {
  BlobSlot *slot = nullptr;
  fcg_status_t st = acquire_slot(lib, &slot);
  if (st != FCG_OK) return st;
  PatchLayout lay;
  st = build_patch_blob(lib, ps, ck, slot->host, BLOB_BYTES, lay);
  if (st != FCG_OK) return st;
  SlotUse use;
  use.slot = slot;
  use.stream = stream;
  FCG_CUDA(cudaMemcpyAsync(slot->dev, slot->host, lay.used, cudaMemcpyHostToDevice, stream));
  use.enqueued = true;
  lib->patch_blob_copy.assign(slot->host, slot->host + lay.used);
  lib->patch_blob_slot = (int)(slot - lib->slots);
  lib->patch_blob_gen = slot->gen;
  lib->patch_blob_stream = consumer;      // the consumer stream is ordered after this upload by the caller (an event wait)
  return FCG_OK;
}

// Host only: would a patch of ps.n_layers layers fit the plan blob and `scratch_limit` bytes of split-KV partials?  The host
// and rope variants ask BEFORE they enqueue their copies / rotation, so that a call that fails has enqueued nothing.
fcg_status_t dry_check_patch(fcg_library *lib, const PatchSpec &ps, const PatchCheck &ck, uint64_t scratch_limit) {
  if (lib->dry_blob.size() < BLOB_BYTES) lib->dry_blob.resize(BLOB_BYTES);
  PatchLayout lay;
  fcg_status_t st = build_patch_blob(lib, ps, ck, lib->dry_blob.data(), BLOB_BYTES, lay);
  if (st != FCG_OK) return st;
  uint64_t po, pm;
  partial_bytes(lib, lay, ps.n_layers, po, pm);
  if (po + pm > scratch_limit)
    return fail(FCG_ERR_OUT_OF_ARENA, "workspace too small for %d-way split partials (%llu bytes) beside the staging area", lay.max_splits,
                (unsigned long long)(po + pm));
  return FCG_OK;
}

// One patch call on device tensors: validate -> blob (uploaded, or the previous call's copy reused) -> growth -> kernels
// -> commit.  `prechecked`: the caller has validated (host / rope variants validate before their own enqueues).
fcg_status_t patch_common(fcg_library *lib, const PatchSpec &ps, const PatchIO &io, const PatchCheck *prechecked = nullptr) {
  fcg_status_t st = validate_io(lib, io);
  if (st != FCG_OK) return st;
  PatchCheck local;
  if (!prechecked) {
    st = validate_patch(lib, ps, local);
    if (st != FCG_OK) return st;
  }
  const PatchCheck &ck = prechecked ? *prechecked : local;

  BlobSlot *slot = nullptr;
  st = acquire_slot(lib, &slot);
  if (st != FCG_OK) return st;
  PatchLayout lay;
  st = build_patch_blob(lib, ps, ck, slot->host, BLOB_BYTES, lay);
  if (st != FCG_OK) return st;
  uint64_t po, pm;
  partial_bytes(lib, lay, io.n_layers, po, pm);
  if (po + pm > lib->scratch_bytes)
    return fail(FCG_ERR_OUT_OF_ARENA, "workspace too small for %d-way split partials (%llu bytes)", lay.max_splits, (unsigned long long)(po + pm));

  SlotUse use;
  use.stream = io.stream;
  {
    const int cached = lib->patch_blob_slot;
    if (cached >= 0 && lib->slots[cached].gen == lib->patch_blob_gen && lib->patch_blob_stream == io.stream &&
        lib->patch_blob_copy.size() == lay.used && memcmp(lib->patch_blob_copy.data(), slot->host, lay.used) == 0) {
      // same bytes as the previous patch call on this stream and its device copy is intact: hand the fresh slot back
      lib->next_slot = (lib->next_slot + BLOB_SLOTS - 1) % BLOB_SLOTS;
      slot->gen--;
      slot = &lib->slots[cached];
      use.slot = slot;
    } else {
      use.slot = slot;
      FCG_CUDA(cudaMemcpyAsync(slot->dev, slot->host, lay.used, cudaMemcpyHostToDevice, io.stream));
      use.enqueued = true;
      lib->patch_blob_copy.assign(slot->host, slot->host + lay.used);
      lib->patch_blob_slot = (int)(slot - lib->slots);
      lib->patch_blob_gen = slot->gen;
      lib->patch_blob_stream = io.stream;
    }
  }
  st = enqueue_growth(lib, lay, slot->dev, io.stream);
  if (st != FCG_OK) return st;
  use.enqueued = true;
  st = launch_patch(lib, lay, slot->dev, io);
  if (st != FCG_OK) return st;
  commit_patch(lib, ps, ck, lay);
  return FCG_OK;
}

}  // namespace

struct fcg_patch_plan {
  fcg_library *lib = nullptr;
  PatchLayout lay;
  uint64_t dev_off = 0, dev_bytes = 0;          // the plan's blob inside the arena (segment allocator)
  std::vector<int32_t> task_ids;
  std::vector<uint32_t> task_gens;
};

fcg_status_t fcg_patch(fcg_library_t *lib, int32_t task_id, int32_t layer_begin, int32_t n_layers, const void *q,
                       const void *k, const void *v, const int32_t *positions, int32_t n, void *out, void *stream) {
  if (!lib) return fail(FCG_ERR_INVALID_ARG, "lib is NULL");
  PatchSpec ps{&task_id, &n, 1, positions, n_layers};
  PatchIO io{layer_begin, n_layers, q, k, v, out, static_cast<cudaStream_t>(stream)};
  FCG_DEVICE(lib);
  FCG_ORDER(lib, io.stream);
  fcg_status_t st = patch_common(lib, ps, io);
  return st != FCG_OK ? st : mark_last(lib, io.stream);
}

fcg_status_t fcg_patch_batch(fcg_library_t *lib, const int32_t *task_ids, const int32_t *n_per_task, int32_t n_tasks,
                             int32_t layer_begin, int32_t n_layers, const void *q, const void *k, const void *v,
                             const int32_t *positions, void *out, void *stream) {
  if (!lib) return fail(FCG_ERR_INVALID_ARG, "lib is NULL");
  PatchSpec ps{task_ids, n_per_task, n_tasks, positions, n_layers};
  PatchIO io{layer_begin, n_layers, q, k, v, out, static_cast<cudaStream_t>(stream)};
  FCG_DEVICE(lib);
  FCG_ORDER(lib, io.stream);
  fcg_status_t st = patch_common(lib, ps, io);
  return st != FCG_OK ? st : mark_last(lib, io.stream);
}

// ------------------------------------------------------------------ patch plans (graph-capturable patching)
fcg_status_t fcg_patch_plan_create(fcg_library_t *lib, const int32_t *task_ids, const int32_t *n_per_task, int32_t n_tasks,
                                   const int32_t *positions, int32_t layers_per_call, void *stream_, fcg_patch_plan_t **out) {
  if (!lib || !out) return fail(FCG_ERR_INVALID_ARG, "NULL argument");
  *out = nullptr;
  if (layers_per_call <= 0 || layers_per_call > lib->cfg.n_layers) return fail(FCG_ERR_INVALID_ARG, "layers_per_call must be in [1, n_layers]");
  cudaStream_t stream = static_cast<cudaStream_t>(stream_);
  PatchSpec ps{task_ids, n_per_task, n_tasks, positions, layers_per_call};
  PatchCheck ck;
  fcg_status_t st = validate_patch(lib, ps, ck);
  if (st != FCG_OK) return st;
  FCG_DEVICE(lib);
  FCG_ORDER(lib, stream);
  BlobSlot *slot = nullptr;
  st = acquire_slot(lib, &slot);
  if (st != FCG_OK) return st;
  fcg_patch_plan *pl = new fcg_patch_plan();
  pl->lib = lib;
  st = build_patch_blob(lib, ps, ck, slot->host, BLOB_BYTES, pl->lay);
  if (st != FCG_OK) {
    delete pl;
    return st;
  }
  {
    uint64_t o_all, ml_all;
    partial_bytes(lib, pl->lay, lib->cfg.n_layers, o_all, ml_all);
    // the slots stay inside the lower half of the scratch area: the upper half is where the host variants stage from their
    // copy stream, and a planned call (possibly a graph replay) cannot record the event that would order them
    if (o_all + ml_all > lib->scratch_total / 2) {
      const int ns = pl->lay.max_splits;
      delete pl;
      return fail(FCG_ERR_OUT_OF_ARENA, "workspace too small for the per-layer partial slots of a %d-way split plan (%llu bytes; a plan may use half of the scratch area)", ns,
                  (unsigned long long)(o_all + ml_all));
    }
  }
  pl->dev_bytes = align_up(pl->lay.used);
  const size_t fi = range_find(lib->seg_free, pl->dev_bytes);
  if (fi == lib->seg_free.size()) {
    delete pl;
    return fail(FCG_ERR_OUT_OF_ARENA, "no free arena range of %llu bytes for a patch plan", (unsigned long long)pl->dev_bytes);
  }
  pl->dev_off = lib->seg_free[fi].off;
  SlotUse use;
  use.slot = slot;
  use.stream = stream;
  cudaError_t e = cudaMemcpyAsync(lib->arena + pl->dev_off, slot->host, pl->lay.used, cudaMemcpyHostToDevice, stream);
  if (e != cudaSuccess) {
    delete pl;
    return fail(FCG_ERR_CUDA, "plan upload: %s", cudaGetErrorString(e));
  }
  use.enqueued = true;
  st = enqueue_growth(lib, pl->lay, lib->arena + pl->dev_off, stream);
  if (st == FCG_OK) st = mark_last(lib, stream);
  if (st != FCG_OK) {
    delete pl;
    return st;
  }
  range_take(lib->seg_free, fi, pl->dev_bytes);
  commit_patch(lib, ps, ck, pl->lay);
  for (int t = 0; t < n_tasks; ++t) {
    pl->task_ids.push_back(task_ids[t]);
    pl->task_gens.push_back(lib->tasks[task_ids[t]].gen);
  }
  lib->n_plans_live++;
  lib->plans.push_back(pl);
  *out = pl;
  return FCG_OK;
}

fcg_status_t fcg_patch_planned(fcg_library_t *lib, fcg_patch_plan_t *plan, int32_t layer_begin, int32_t n_layers, const void *q,
                               const void *k, const void *v, void *out, void *stream_) {
  // membership first: a destroyed plan (or one of another library) is recognised without touching its memory
  if (!lib || !plan || std::find(lib->plans.begin(), lib->plans.end(), plan) == lib->plans.end())
    return fail(FCG_ERR_INVALID_ARG, "NULL plan, a plan of another library or one that was already destroyed");
  for (size_t t = 0; t < plan->task_ids.size(); ++t) {
    const TaskRec &tr = lib->tasks[plan->task_ids[t]];
    if (!tr.live || tr.gen != plan->task_gens[t])
      return fail(FCG_ERR_BAD_TASK, "task %d was released or re-stitched after the plan was made", plan->task_ids[t]);
  }
  if ((int64_t)n_layers * (int64_t)plan->task_ids.size() > 65535)
    return fail(FCG_ERR_INVALID_ARG, "%d layers x %zu tasks in one call exceed the launch limit of 65535", n_layers, plan->task_ids.size());
  PatchIO io{layer_begin, n_layers, q, k, v, out, static_cast<cudaStream_t>(stream_)};
  fcg_status_t st = validate_io(lib, io);
  if (st != FCG_OK) return st;
  FCG_DEVICE(lib);
  bool capturing = false;
  st = order_after_previous(lib, io.stream, &capturing);
  if (st != FCG_OK) return st;
  st = launch_patch(lib, plan->lay, lib->arena + plan->dev_off, io, /*layer_slots=*/true);
  if (st != FCG_OK) return st;
  return capturing ? FCG_OK : mark_last(lib, io.stream);
}

fcg_status_t fcg_patch_plan_destroy(fcg_library_t *lib, fcg_patch_plan_t *plan) {
  if (!lib || !plan) return fail(FCG_ERR_INVALID_ARG, "NULL library / plan");
  auto it = std::find(lib->plans.begin(), lib->plans.end(), plan);   // before the plan's memory is touched (found by the ASan run)
  if (it == lib->plans.end()) return fail(FCG_ERR_INVALID_ARG, "a plan of another library or one that was already destroyed");
  lib->plans.erase(it);
  range_give(lib->seg_free, plan->dev_off, plan->dev_bytes);
  lib->n_plans_live--;
  delete plan;
  return FCG_OK;
}

// fcg_library_destroy: plans the caller never destroyed go with the library
extern "C++" void free_plans(fcg_library *lib) {
  for (fcg_patch_plan *pl : lib->plans) delete pl;
  lib->plans.clear();
  lib->n_plans_live = 0;
}

// NEXT-4 (R13 variant): q and k arrive before position encoding; rotate them to positions[i], then patch
fcg_status_t fcg_patch_rope(fcg_library_t *lib, int32_t task_id, int32_t layer_begin, int32_t n_layers, const void *q,
                            const void *k, const void *v, const int32_t *positions, int32_t n, void *out, void *stream_) {
  if (!lib) return fail(FCG_ERR_INVALID_ARG, "lib is NULL");
  const fcg_config_t &c = lib->cfg;
  if (c.rope_mode == FCG_ROPE_NONE) return fcg_patch(lib, task_id, layer_begin, n_layers, q, k, v, positions, n, out, stream_);
  cudaStream_t stream = static_cast<cudaStream_t>(stream_);
  // every host-side check first: nothing is enqueued for a call that fails (fcg.h conventions)
  PatchSpec ps{&task_id, &n, 1, positions, n_layers};
  PatchIO io0{layer_begin, n_layers, q, k, v, out, stream};
  fcg_status_t st = validate_io(lib, io0);
  if (st != FCG_OK) return st;
  PatchCheck ck;
  st = validate_patch(lib, ps, ck);
  if (st != FCG_OK) return st;
  const int half = c.head_dim / 2;
  const uint64_t q_bytes = (uint64_t)n_layers * n * c.n_q_heads * c.head_dim * 2;
  const uint64_t kv_bytes = (uint64_t)n_layers * n * c.n_kv_heads * c.head_dim * 2;
  const uint64_t tab_bytes = (uint64_t)n * half * sizeof(float4);
  const uint64_t need = align_up(q_bytes) + align_up(kv_bytes);
  if (tab_bytes > BLOB_BYTES) return fail(FCG_ERR_OUT_OF_ARENA, "rope table of %d tokens exceeds the %llu-byte plan blob", n, (unsigned long long)BLOB_BYTES);
  if (need > lib->scratch_bytes / 2) return fail(FCG_ERR_OUT_OF_ARENA, "workspace too small for %llu bytes of rotated q / k", (unsigned long long)need);
  // rotated copies at the END of the scratch area (where fcg_patch_host stages too); split partials grow from its start
  unsigned char *dq = lib->arena + lib->scratch_off + lib->scratch_bytes - need, *dk = dq + align_up(q_bytes);
  st = dry_check_patch(lib, ps, ck, lib->scratch_bytes - need);
  if (st != FCG_OK) return st;

  FCG_DEVICE(lib);
  FCG_ORDER(lib, stream);
  BlobSlot *slot = nullptr;
  st = acquire_slot(lib, &slot);
  if (st != FCG_OK) return st;
  SlotUse use;
  use.slot = slot;
  use.stream = stream;
  // cos / sin of p_i * theta_j in fp64: exact evaluation at the start of every run of consecutive positions (and every
  // 32 tokens), angle addition by theta_j in between (error ~1e-16 per step), then the hi / lo split of the stitch table
  float4 *tab = reinterpret_cast<float4 *>(slot->host);
  std::vector<double> cs(half), sn(half), c1(half), s1(half);
  for (int j = 0; j < half; ++j) {
    c1[j] = cos(lib->inv_freq[j]);
    s1[j] = sin(lib->inv_freq[j]);
  }
  auto split = [](double x, float &hi, float &lo) {
    float f = (float)x;
    uint32_t b;
    memcpy(&b, &f, 4);
    b = (b + 0x80u) & 0xffffff00u;
    memcpy(&hi, &b, 4);
    lo = (float)(x - (double)hi);
  };
  for (int i = 0, run = 0; i < n; ++i) {
    const bool anchor = i == 0 || positions[i] != positions[i - 1] + 1 || run >= 32;
    for (int j = 0; j < half; ++j) {
      if (anchor) {
        const double phi = (double)positions[i] * lib->inv_freq[j];
        cs[j] = cos(phi);
        sn[j] = sin(phi);
      } else {
        const double cn = cs[j] * c1[j] - sn[j] * s1[j], snn = sn[j] * c1[j] + cs[j] * s1[j];
        cs[j] = cn;
        sn[j] = snn;
      }
      float4 t;
      split(cs[j], t.x, t.y);
      split(sn[j], t.z, t.w);
      tab[(size_t)i * half + j] = t;
    }
    run = anchor ? 0 : run + 1;
  }
  FCG_CUDA(cudaMemcpyAsync(slot->dev, slot->host, tab_bytes, cudaMemcpyHostToDevice, stream));
  use.enqueued = true;
  fcg::RopeQkParams rp;
  rp.q = static_cast<const uint16_t *>(q);
  rp.k = static_cast<const uint16_t *>(k);
  rp.q_out = reinterpret_cast<uint16_t *>(dq);
  rp.k_out = reinterpret_cast<uint16_t *>(dk);
  rp.table = reinterpret_cast<const float4 *>(slot->dev);
  rp.n_layers = n_layers;
  rp.n_total = n;
  rp.n_q_heads = c.n_q_heads;
  rp.n_kv_heads = c.n_kv_heads;
  rp.interleaved = c.rope_mode == FCG_ROPE_INTERLEAVED ? 1 : 0;
  rp.head_dim = c.head_dim;
  FCG_CUDA(fcg::launch_rope_qk(rp, c.head_dim, stream));
  lib->stats.rope_qk_launches++;
  const uint64_t saved = lib->scratch_bytes;
  lib->scratch_bytes = saved - need;
  PatchIO io{layer_begin, n_layers, dq, dk, v, out, stream};
  st = patch_common(lib, ps, io, &ck);
  lib->scratch_bytes = saved;
  if (cudaEventRecord(lib->staging_ev, stream) == cudaSuccess) lib->have_staging_ev = true;   // dq / dk are in use until here
  fcg_status_t mst = mark_last(lib, stream);
  return st != FCG_OK ? st : mst;
}

}  // extern "C"

namespace {
// host-buffer patch of one task or of a batch: n = total patch tokens over the tasks
fcg_status_t patch_host_common(fcg_library *lib, const int32_t *task_ids, const int32_t *n_per_task, int32_t n_tasks,
                               int32_t layer_begin, int32_t n_layers, const void *q, const void *k, const void *v,
                               const int32_t *positions, void *out, void *stream_) {
  const fcg_config_t &c = lib->cfg;
  cudaStream_t stream = static_cast<cudaStream_t>(stream_);
  // every host-side check first: nothing is copied or launched for a call that fails (fcg.h conventions)
  PatchIO io0{layer_begin, n_layers, q, k, v, out, stream};
  fcg_status_t st = validate_io(lib, io0);
  if (st != FCG_OK) return st;
  PatchSpec ps0{task_ids, n_per_task, n_tasks, positions, n_layers};
  PatchCheck ck;
  st = validate_patch(lib, ps0, ck);
  if (st != FCG_OK) return st;
  const int64_t n = ck.n_total;
  const uint64_t q_bytes = (uint64_t)n_layers * n * c.n_q_heads * c.head_dim * 2;
  const uint64_t kv_bytes = (uint64_t)n_layers * n * c.n_kv_heads * c.head_dim * 2;
  const uint64_t need = 2 * align_up(q_bytes) + 2 * align_up(kv_bytes);
  // staging sits at the END of the scratch area; split partials grow from its start
  if (need > lib->scratch_bytes / 2) return fail(FCG_ERR_OUT_OF_ARENA, "workspace too small to stage %llu bytes", (unsigned long long)need);
  unsigned char *base = lib->arena + lib->scratch_off + lib->scratch_bytes - need;
  unsigned char *dq = base, *dk = dq + align_up(q_bytes), *dv = dk + align_up(kv_bytes), *dout = dv + align_up(kv_bytes);
  {
    // the largest layer group decides (the split choice and the partials grow with the layers of one call)
    const int groups_ = (q_bytes >= (8ull << 20) && n_layers >= fcg_library::HOST_GROUPS) ? fcg_library::HOST_GROUPS : 1;
    int max_nl = 0;
    for (int g = 0; g < groups_; ++g) max_nl = std::max(max_nl, (int)((int64_t)n_layers * (g + 1) / groups_) - (int)((int64_t)n_layers * g / groups_));
    PatchSpec ps_max{task_ids, n_per_task, n_tasks, positions, max_nl};
    st = dry_check_patch(lib, ps_max, ck, lib->scratch_bytes - need);
    if (st != FCG_OK) return st;
  }
  FCG_DEVICE(lib);
  FCG_ORDER(lib, stream);
  // Copies in on the library's copy stream: after the last user of the staging area (staging_ev: host and rope calls),
  // but NOT after a stitch the caller has just enqueued on `stream` (stitch never touches the scratch area), so the
  // host->device copies overlap it.  Large calls are cut into layer groups: group g attends while group g+1 is still
  // arriving and group g-1 is leaving (second copy stream), all joined back into `stream` at the end.
  const int groups = (q_bytes >= (8ull << 20) && n_layers >= fcg_library::HOST_GROUPS) ? fcg_library::HOST_GROUPS : 1;
  const uint64_t q_layer = q_bytes / n_layers, kv_layer = kv_bytes / n_layers;
  auto group_begin = [&](int g) { return (int)((int64_t)n_layers * g / groups); };
  if (lib->have_staging_ev) FCG_CUDA(cudaStreamWaitEvent(lib->copy_stream, lib->staging_ev, 0));
  {
    // the first group's plan blob goes ahead of the big copies, on the copy stream (prime_patch_blob): `stream` picks it
    // up through h2d_ev[0]; on `stream` itself it would sit behind the caller's stitch and block the copy queue
    PatchSpec ps_g0{task_ids, n_per_task, n_tasks, positions, group_begin(1) - group_begin(0)};
    st = prime_patch_blob(lib, ps_g0, ck, lib->copy_stream, stream);
    if (st != FCG_OK) return st;
  }
  for (int g = 0; g < groups; ++g) {
    const int lb = group_begin(g), nl = group_begin(g + 1) - lb;
    FCG_CUDA(cudaMemcpyAsync(dq + lb * q_layer, (const char *)q + lb * q_layer, nl * q_layer, cudaMemcpyHostToDevice, lib->copy_stream));
    FCG_CUDA(cudaMemcpyAsync(dk + lb * kv_layer, (const char *)k + lb * kv_layer, nl * kv_layer, cudaMemcpyHostToDevice, lib->copy_stream));
    FCG_CUDA(cudaMemcpyAsync(dv + lb * kv_layer, (const char *)v + lb * kv_layer, nl * kv_layer, cudaMemcpyHostToDevice, lib->copy_stream));
    FCG_CUDA(cudaEventRecord(lib->h2d_ev[g], lib->copy_stream));
  }
  // partials must not collide with the staging area: temporarily shrink the scratch
  const uint64_t saved = lib->scratch_bytes;
  lib->scratch_bytes = saved - need;
  for (int g = 0; g < groups && st == FCG_OK; ++g) {
    const int lb = group_begin(g), nl = group_begin(g + 1) - lb;
    cudaError_t e = cudaStreamWaitEvent(stream, lib->h2d_ev[g], 0);
    if (e != cudaSuccess) {
      st = fail(FCG_ERR_CUDA, "cudaStreamWaitEvent: %s", cudaGetErrorString(e));
      break;
    }
    PatchSpec ps{task_ids, n_per_task, n_tasks, positions, nl};
    PatchIO io{layer_begin + lb, nl, dq + lb * q_layer, dk + lb * kv_layer, dv + lb * kv_layer, dout + lb * q_layer, stream};
    // group 0 carries the growth (if any) and commits the fill state; the later groups re-validate against it (cheap)
    st = patch_common(lib, ps, io, g == 0 ? &ck : nullptr);
    if (st != FCG_OK) break;
    if (groups > 1) {
      e = cudaEventRecord(lib->attn_ev[g], stream);
      if (e == cudaSuccess) e = cudaStreamWaitEvent(lib->d2h_stream, lib->attn_ev[g], 0);
      if (e == cudaSuccess)
        e = cudaMemcpyAsync((char *)out + lb * q_layer, dout + lb * q_layer, nl * q_layer, cudaMemcpyDeviceToHost, lib->d2h_stream);
      if (e != cudaSuccess) st = fail(FCG_ERR_CUDA, "copy out: %s", cudaGetErrorString(e));
    }
  }
  lib->scratch_bytes = saved;
  if (st == FCG_OK) {
    cudaError_t e = cudaSuccess;
    if (groups > 1) {
      e = cudaEventRecord(lib->d2h_ev, lib->d2h_stream);
      if (e == cudaSuccess) e = cudaStreamWaitEvent(stream, lib->d2h_ev, 0);
    } else {
      e = cudaMemcpyAsync(out, dout, q_bytes, cudaMemcpyDeviceToHost, stream);
    }
    if (e != cudaSuccess) st = fail(FCG_ERR_CUDA, "copy out: %s", cudaGetErrorString(e));
  }
  // the copy streams have work in flight whatever happened above: `stream` joins them, and the next user of the staging
  // area waits for this point
  cudaStreamWaitEvent(stream, lib->h2d_ev[groups - 1], 0);
  if (cudaEventRecord(lib->staging_ev, stream) == cudaSuccess) lib->have_staging_ev = true;
  fcg_status_t mst = mark_last(lib, stream);
  return st != FCG_OK ? st : mst;
}
}  // namespace

extern "C" {

fcg_status_t fcg_patch_host(fcg_library_t *lib, int32_t task_id, int32_t layer_begin, int32_t n_layers, const void *q,
                            const void *k, const void *v, const int32_t *positions, int32_t n, void *out, void *stream) {
  if (!lib) return fail(FCG_ERR_INVALID_ARG, "lib is NULL");
  return patch_host_common(lib, &task_id, &n, 1, layer_begin, n_layers, q, k, v, positions, out, stream);
}

fcg_status_t fcg_patch_batch_host(fcg_library_t *lib, const int32_t *task_ids, const int32_t *n_per_task, int32_t n_tasks,
                                  int32_t layer_begin, int32_t n_layers, const void *q, const void *k, const void *v,
                                  const int32_t *positions, void *out, void *stream) {
  if (!lib) return fail(FCG_ERR_INVALID_ARG, "lib is NULL");
  return patch_host_common(lib, task_ids, n_per_task, n_tasks, layer_begin, n_layers, q, k, v, positions, out, stream);
}

// ------------------------------------------------------------------------------- task utilities
fcg_status_t fcg_task_page_table(fcg_library_t *lib, int32_t task_id, const int32_t **dev_table, int32_t *n_pages,
                                 int32_t *n_tokens) {
  if (!lib) return fail(FCG_ERR_INVALID_ARG, "lib is NULL");
  if (task_id < 0 || task_id >= lib->cfg.max_tasks || !lib->tasks[task_id].live) return fail(FCG_ERR_BAD_TASK, "unknown task %d", task_id);
  const TaskRec &t = lib->tasks[task_id];
  if (dev_table) *dev_table = lib->tables() + (int64_t)task_id * lib->pages_per_task;
  if (n_pages) *n_pages = (int32_t)t.pages.size();
  if (n_tokens) *n_tokens = t.n_tokens;
  return FCG_OK;
}

fcg_status_t fcg_task_page_table_host(fcg_library_t *lib, int32_t task_id, int32_t *out, int32_t cap, int32_t *n_pages) {
  if (!lib) return fail(FCG_ERR_INVALID_ARG, "lib is NULL");
  if (task_id < 0 || task_id >= lib->cfg.max_tasks || !lib->tasks[task_id].live) return fail(FCG_ERR_BAD_TASK, "unknown task %d", task_id);
  const TaskRec &t = lib->tasks[task_id];
  if (n_pages) *n_pages = (int32_t)t.pages.size();
  if (out && cap > 0) memcpy(out, t.pages.data(), sizeof(int32_t) * std::min<size_t>(cap, t.pages.size()));
  return FCG_OK;
}

fcg_status_t fcg_task_boundary_positions(fcg_library_t *lib, int32_t task_id, int32_t width, int32_t *out, int32_t cap,
                                         int32_t *n_out) {
  if (!lib || !n_out) return fail(FCG_ERR_INVALID_ARG, "NULL argument");
  if (task_id < 0 || task_id >= lib->cfg.max_tasks || !lib->tasks[task_id].live) return fail(FCG_ERR_BAD_TASK, "unknown task %d", task_id);
  if (width <= 0) return fail(FCG_ERR_INVALID_ARG, "width must be > 0");
  std::vector<int32_t> pos;
  for (auto &sp : lib->tasks[task_id].spans)
    if (sp.first > 0)
      for (int32_t x = sp.first; x < sp.first + std::min(width, sp.second); ++x) pos.push_back(x);
  std::sort(pos.begin(), pos.end());
  pos.erase(std::unique(pos.begin(), pos.end()), pos.end());
  *n_out = (int32_t)pos.size();
  if (out && cap > 0) memcpy(out, pos.data(), sizeof(int32_t) * std::min<size_t>(cap, pos.size()));
  return FCG_OK;
}

fcg_status_t fcg_task_release(fcg_library_t *lib, int32_t task_id) {
  if (!lib) return fail(FCG_ERR_INVALID_ARG, "lib is NULL");
  if (task_id < 0 || task_id >= lib->cfg.max_tasks || !lib->tasks[task_id].live) return fail(FCG_ERR_BAD_TASK, "unknown task %d", task_id);
  TaskRec &t = lib->tasks[task_id];
  for (auto it = t.pages.rbegin(); it != t.pages.rend(); ++it) lib->page_stack.push_back(*it);
  t = TaskRec();
  t.gen = ++lib->task_gen;
  lib->n_tasks_live--;
  return FCG_OK;
}

// ------------------------------------------------------------- NEXT-1: suffix re-graft (Eq. 6)
fcg_status_t fcg_task_shift(fcg_library_t *lib, int32_t task_id, int32_t src_begin, int32_t n_tokens, int32_t dst_begin,
                            void *stream_) {
  if (!lib) return fail(FCG_ERR_INVALID_ARG, "lib is NULL");
  const fcg_config_t &c = lib->cfg;
  if (task_id < 0 || task_id >= c.max_tasks || !lib->tasks[task_id].live) return fail(FCG_ERR_BAD_TASK, "unknown task %d", task_id);
  TaskRec &t = lib->tasks[task_id];
  if (n_tokens <= 0 || src_begin < 0 || dst_begin < 0 || (int64_t)src_begin + n_tokens > t.capacity ||
      (int64_t)dst_begin + n_tokens > c.max_task_tokens)
    return fail(FCG_ERR_RANGE, "shift source outside the capacity %d of task %d, or destination outside max_task_tokens %d", t.capacity,
                task_id, c.max_task_tokens);
  for (int32_t x = src_begin; x < src_begin + n_tokens; ++x)
    if (!t.filled[x]) return fail(FCG_ERR_UNFILLED, "task %d: shift source position %d was never filled", task_id, x);
  const int32_t delta = dst_begin - src_begin;
  if (delta == 0) return FCG_OK;
  cudaStream_t stream = static_cast<cudaStream_t>(stream_);
  const int P = c.page_size;
  const int32_t dst_end = dst_begin + n_tokens;
  const int32_t n_old = (int32_t)t.pages.size();
  // R25: every logical page that receives a new physical page -- gap pages between the end of the table and the
  // destination (a destination beyond the capacity appends), then the destination's pages -- ascending logical order
  const int32_t lp0 = dst_begin / P, lp1 = (dst_end - 1) / P, first_new = std::min(lp0, n_old), n_new = lp1 - first_new + 1;
  if ((size_t)n_new > lib->page_stack.size())
    return fail(FCG_ERR_OUT_OF_PAGES, "need %d pages, %zu free", n_new, lib->page_stack.size());
  const int32_t new_cap = std::max(t.capacity, dst_end);

  // copy-on-shift: destination pages are fresh, so no page is read and written by the same launch
  GatherBuilder gb;
  std::vector<int32_t> stack = lib->page_stack;
  for (int32_t k = 0; k < n_new; ++k) {
    gb.pages.push_back(stack.back());
    stack.pop_back();
  }
  fcg::StitchEntryDev de;
  gb.pool_side(lib, de.k_src, de.v_src, de.src_layer_stride, de.src_head_stride);
  gb.pool_side(lib, de.k_dst, de.v_dst, de.dst_layer_stride, de.dst_head_stride);
  de.src_fp8 = 0;
  de.k_exp = de.v_exp = 0;
  de.table_off = gb.table_for(lib, delta);
  gb.entries.push_back(de);          // entry 0: the moved range, rotated by delta
  de.table_off = -1;
  gb.entries.push_back(de);          // entry 1: the other slots of the re-paged pages, bit copy
  auto add_chunk = [&](int32_t entry, int32_t dst_pos, int32_t src_pos, int32_t n) {
    fcg::StitchChunkDev dc;
    dc.entry = entry;
    dc.dst_tok = gb.pool_tok(lib, gb.pages[dst_pos / P - first_new], dst_pos % P);
    dc.src_tok = gb.pool_tok(lib, t.pages[src_pos / P], src_pos % P);
    dc.ntok = n;
    gb.chunks.push_back(dc);
  };
  for (int32_t done = 0; done < n_tokens;) {          // runs contiguous in one source page and one destination page
    const int32_t d = dst_begin + done, sp = src_begin + done;
    const int32_t n = std::min(std::min(P - d % P, P - sp % P), n_tokens - done);
    add_chunk(0, d, sp, n);
    done += n;
  }
  // slots of re-paged pages outside the destination keep their contents -- as far as the old table held them
  const int32_t old_end = std::min(n_old * P, t.capacity);
  if (dst_begin > lp0 * P && lp0 * P < old_end) add_chunk(1, lp0 * P, lp0 * P, std::min(dst_begin, old_end) - lp0 * P);
  const int32_t page_end = std::min((lp1 + 1) * P, old_end);
  if (dst_end < page_end) add_chunk(1, dst_end, dst_end, page_end - dst_end);

  FCG_DEVICE(lib);
  FCG_ORDER(lib, stream);
  GatherBlob gbl;
  fcg_status_t st = enqueue_gather(lib, gb, stream, gbl);
  if (st != FCG_OK) return st;
  FCG_CUDA(cudaMemcpyAsync(lib->tables() + (int64_t)task_id * lib->pages_per_task + first_new, gbl.slot->dev + gbl.off_pages,
                           (size_t)n_new * sizeof(int32_t), cudaMemcpyDeviceToDevice, stream));
  st = mark_last(lib, stream);
  if (st != FCG_OK) return st;

  // ---- commit: new pages in, replaced pages back to the pool (re-issued in ascending logical order) ----
  lib->page_stack.swap(stack);
  for (int32_t lp = std::min(lp1, n_old - 1); lp >= lp0; --lp) lib->page_stack.push_back(t.pages[lp]);
  if ((int32_t)t.pages.size() < lp1 + 1) t.pages.resize(lp1 + 1);
  for (int32_t lp = first_new; lp <= lp1; ++lp) t.pages[lp] = gb.pages[lp - first_new];
  if (new_cap > t.capacity) {
    t.capacity = new_cap;
    t.filled.resize(new_cap, 0);
  }
  std::fill(t.filled.begin() + src_begin, t.filled.begin() + src_begin + n_tokens, (uint8_t)0);
  std::fill(t.filled.begin() + dst_begin, t.filled.begin() + dst_end, (uint8_t)1);
  t.filled_prefix = 0;
  while (t.filled_prefix < t.capacity && t.filled[t.filled_prefix]) t.filled_prefix++;
  t.n_tokens = std::max(t.n_tokens, dst_end);
  // positions were un-filled and pages re-assigned: a patch plan made before the shift no longer describes this task
  // (fcg_patch_planned does not re-validate the fill state, it compares generations)
  t.gen = ++lib->task_gen;
  return FCG_OK;
}

// ------------------------------------------------------- NEXT-2: segment extraction (Alg. 1B update)
fcg_status_t fcg_segment_extract(fcg_library_t *lib, int32_t task_id, int32_t begin, int32_t n_tokens, int32_t new_orig_start,
                                 void *stream_, int32_t *seg_id_out) {
  if (!lib || !seg_id_out) return fail(FCG_ERR_INVALID_ARG, "NULL argument");
  const fcg_config_t &c = lib->cfg;
  if (task_id < 0 || task_id >= c.max_tasks || !lib->tasks[task_id].live) return fail(FCG_ERR_BAD_TASK, "unknown task %d", task_id);
  const TaskRec &t = lib->tasks[task_id];
  if (n_tokens <= 0 || begin < 0 || (int64_t)begin + n_tokens > t.capacity)
    return fail(FCG_ERR_RANGE, "extract range outside the capacity %d of task %d", t.capacity, task_id);
  if (new_orig_start < 0) return fail(FCG_ERR_INVALID_ARG, "new_orig_start must be >= 0");
  for (int32_t x = begin; x < begin + n_tokens; ++x)
    if (!t.filled[x]) return fail(FCG_ERR_UNFILLED, "task %d: extract position %d was never filled", task_id, x);
  SegmentSlot sl;
  fcg_status_t st = find_segment_slot(lib, n_tokens, sl);
  if (st != FCG_OK) return st;
  cudaStream_t stream = static_cast<cudaStream_t>(stream_);
  const int P = c.page_size;

  GatherBuilder gb;
  fcg::StitchEntryDev de;
  gb.pool_side(lib, de.k_src, de.v_src, de.src_layer_stride, de.src_head_stride);
  gb.segment_side(lib, lib->arena, sl.off, sl.bytes, n_tokens, de.k_dst, de.v_dst, de.dst_layer_stride, de.dst_head_stride);
  de.table_off = gb.table_for(lib, new_orig_start - begin);
  de.src_fp8 = 0;
  de.k_exp = de.v_exp = 0;
  gb.entries.push_back(de);
  for (int32_t done = 0; done < n_tokens;) {          // one chunk per source page
    const int32_t sp = begin + done;
    const int32_t n = std::min(P - sp % P, n_tokens - done);
    fcg::StitchChunkDev dc;
    dc.entry = 0;
    dc.dst_tok = done;
    dc.src_tok = gb.pool_tok(lib, t.pages[sp / P], sp % P);
    dc.ntok = n;
    gb.chunks.push_back(dc);
    done += n;
  }
  FCG_DEVICE(lib);
  FCG_ORDER(lib, stream);
  GatherBlob gbl;
  st = enqueue_gather(lib, gb, stream, gbl);
  if (st != FCG_OK) return st;
  st = mark_last(lib, stream);
  if (st != FCG_OK) return st;
  commit_segment_slot(lib, sl, n_tokens, new_orig_start);
  *seg_id_out = sl.sid;
  return FCG_OK;
}

fcg_status_t fcg_task_read(fcg_library_t *lib, int32_t task_id, int32_t layer, int32_t begin, int32_t n, void *k_out,
                           void *v_out, void *stream) {
  if (!lib || !k_out || !v_out) return fail(FCG_ERR_INVALID_ARG, "NULL argument");
  const fcg_config_t &c = lib->cfg;
  if (task_id < 0 || task_id >= c.max_tasks || !lib->tasks[task_id].live) return fail(FCG_ERR_BAD_TASK, "unknown task %d", task_id);
  const TaskRec &t = lib->tasks[task_id];
  if (layer < 0 || layer >= c.n_layers) return fail(FCG_ERR_INVALID_ARG, "layer out of range");
  if (begin < 0 || n <= 0 || (int64_t)begin + n > t.capacity) return fail(FCG_ERR_RANGE, "token range outside capacity");
  fcg::ReadParams rp;
  rp.k_pool = lib->k_pool();
  rp.v_pool = lib->v_pool();
  rp.k_out = static_cast<uint16_t *>(k_out);
  rp.v_out = static_cast<uint16_t *>(v_out);
  rp.table = lib->tables() + (int64_t)task_id * lib->pages_per_task;
  rp.layer = layer;
  rp.begin = begin;
  rp.n = n;
  rp.n_kv_heads = c.n_kv_heads;
  rp.head_dim = c.head_dim;
  rp.page_size = c.page_size;
  rp.n_pages = c.n_pages;
  FCG_DEVICE(lib);
  FCG_ORDER(lib, static_cast<cudaStream_t>(stream));
  FCG_CUDA(fcg::launch_task_read(rp, static_cast<cudaStream_t>(stream)));
  lib->stats.read_launches++;
  return mark_last(lib, static_cast<cudaStream_t>(stream));
}

fcg_status_t fcg_pool_info(fcg_library_t *lib, fcg_pool_info_t *out) {
  if (!lib || !out) return fail(FCG_ERR_INVALID_ARG, "NULL argument");
  out->k_pool_offset = lib->k_pool_off;
  out->v_pool_offset = lib->v_pool_off;
  out->pool_bytes = lib->pool_bytes;
  out->page_table_offset = lib->table_off;
  out->workspace_offset = lib->ws_off;
  out->segments_offset = lib->seg_off;
  uint64_t fr = 0;
  for (auto &r : lib->seg_free) fr += r.bytes;
  out->segments_bytes_free = fr;
  out->n_pages = lib->cfg.n_pages;
  out->n_pages_free = (uint32_t)lib->page_stack.size();
  out->n_segments_live = lib->n_segments_live;
  out->n_tasks_live = lib->n_tasks_live;
  return FCG_OK;
}

fcg_status_t fcg_set_attn_policy(fcg_library_t *lib, int32_t tc_min_rows, int32_t force_splits) {
  if (!lib || tc_min_rows < 0 || force_splits < 0) return fail(FCG_ERR_INVALID_ARG, "NULL library or negative threshold / split count");
  lib->tc_min_rows = tc_min_rows;
  lib->force_splits = force_splits;
  return FCG_OK;
}

fcg_status_t fcg_set_attn_mixed(fcg_library_t *lib, int32_t enable) {
  if (!lib) return fail(FCG_ERR_INVALID_ARG, "lib is NULL");
  lib->mix_classes = enable != 0;
  return FCG_OK;
}

fcg_status_t fcg_set_attn_pairs(fcg_library_t *lib, int32_t enable) {
  if (!lib) return fail(FCG_ERR_INVALID_ARG, "lib is NULL");
  lib->use_pairs = enable != 0;
  return FCG_OK;
}

fcg_status_t fcg_stats(fcg_library_t *lib, fcg_stats_t *out) {
  if (!lib || !out) return fail(FCG_ERR_INVALID_ARG, "NULL argument");
  *out = lib->stats;
  return FCG_OK;
}

}  // extern "C"
