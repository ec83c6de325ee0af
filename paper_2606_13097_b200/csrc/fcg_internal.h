// Internal declarations shared by the host side (fcg_api.cu) and the kernels of libfcg.so.
// Not part of the public ABI (that is include/fcg.h).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

namespace fcg {

// sets the thread-local message behind fcg_last_error() (defined in fcg_api.cu)
void set_last_error(const char *msg);

// ---------------------------------------------------------------------------------------------
// S3: fused gather + RoPE-shift.  One kernel moves token rows between any two of {library segment,
// paged cache}: stitch (segment -> cache), suffix re-graft (cache -> cache, fcg_task_shift) and segment
// extraction (cache -> segment).  An entry fixes source, destination and the rotation; a chunk is a run
// of consecutive token rows of one entry that is contiguous on both sides (at most one page).
// Row address of (layer, kv head g, token t) = base + (layer * layer_stride + g * head_stride + tok + t) * D * 2:
//   segment [L][Hkv][n][D]:          layer_stride = Hkv * n,           head_stride = n, tok = index in the segment
//   pool    [L][n_pages][Hkv][P][D]: layer_stride = n_pages * Hkv * P, head_stride = P, tok = page * Hkv * P + slot
// ---------------------------------------------------------------------------------------------
struct StitchEntryDev {  // 80 B
  uint64_t k_src, v_src;         // device addresses of the source K / V (bf16 rows, or e4m3 code rows: src_fp8)
  uint64_t k_dst, v_dst;         // device addresses of the destination K / V
  int64_t src_layer_stride;      // in token rows
  int64_t dst_layer_stride;
  int32_t src_head_stride;
  int32_t dst_head_stride;
  int32_t table_off;             // first float4 of this entry's rope table; -1 -> bit copy (delta 0 / rope off)
  int32_t src_fp8;               // 1: the source is an fp8 segment (R26): D code bytes per row + one scale byte per row
  uint64_t k_exp, v_exp;         // fp8 source: device addresses of the per-row scale exponents (one byte e + 127 per row)
};

struct StitchChunkDev {  // 16 B
  int32_t entry;         // index into the entry array
  int32_t dst_tok;       // destination row offset of the chunk's first token (see above)
  int32_t src_tok;       // source row offset of the chunk's first token
  int32_t ntok;          // tokens in the chunk
};

struct StitchParams {
  int32_t any_fp8;       // some entry reads an fp8 segment: launch the kernel variant that can de-quantise
  const StitchEntryDev *entries;
  const StitchChunkDev *chunks;
  const float4 *table;   // per (entry, j): {c_hi, c_lo, s_hi, s_lo}; c_hi/s_hi have <= 16 significant bits
  int32_t n_chunks, n_layers, n_kv_heads;
  int32_t interleaved;   // 0: pairs (j, j + D/2) (half-split); 1: pairs (2j, 2j + 1)
  int32_t head_dim;      // row length in elements (the run-time-D instantiation reads it)
};

cudaError_t launch_stitch(const StitchParams &p, int head_dim, cudaStream_t stream);

// fcg_patch_rope: rotate the patch's q and k rows (given before position encoding) to their absolute positions.
// table: per (token i, j): {c_hi, c_lo, s_hi, s_lo} of p_i * theta_j, same split as the stitch table.
struct RopeQkParams {
  const uint16_t *q, *k;     // [n_layers][n_total][Hq | Hkv][D]
  uint16_t *q_out, *k_out;   // same shapes
  const float4 *table;       // [n_total][D/2]
  int32_t n_layers, n_total, n_q_heads, n_kv_heads, interleaved;
  int32_t head_dim;
};
cudaError_t launch_rope_qk(const RopeQkParams &p, int head_dim, cudaStream_t stream);

// ---------------------------------------------------------------------------------------------
// S1 (register copy), S4 (scatter), task read
// ---------------------------------------------------------------------------------------------
struct RegisterParams {
  const uint16_t *k_src, *v_src;
  uint16_t *k_dst, *v_dst;   // contiguous [L][Hkv][n][D]
  int64_t s_layer, s_head, s_tok;  // source strides in elements
  int32_t n_layers, n_kv_heads, n_tokens, head_dim;
};
cudaError_t launch_register_copy(const RegisterParams &p, cudaStream_t stream);
// S1 with fp8 storage (R26): quantise the caller's bf16 rows to e4m3 codes + one power-of-two scale exponent per row.
// k_dst / v_dst: [L][Hkv][n][D] bytes; k_exp / v_exp: [L][Hkv][n] bytes (e + 127)
struct RegisterFp8Params {
  const uint16_t *k_src, *v_src;
  uint8_t *k_dst, *v_dst, *k_exp, *v_exp;
  int64_t s_layer, s_head, s_tok;  // source strides in elements
  int32_t n_layers, n_kv_heads, n_tokens, head_dim;
};
cudaError_t launch_register_fp8(const RegisterFp8Params &p, cudaStream_t stream);

struct ScatterParams {
  const uint16_t *k_new, *v_new;  // [n_layers][n_total][Hkv][D]
  uint16_t *k_pool, *v_pool;
  const int32_t *tables;          // page-table region
  const int32_t *positions;       // [n_total]
  const int32_t *tok_table_off;   // [n_total] page-table offset of the token's task
  int32_t n_layers, layer_begin, n_total, n_kv_heads, head_dim, page_size;
  uint32_t n_pages;
};
cudaError_t launch_scatter(const ScatterParams &p, cudaStream_t stream);

struct ReadParams {
  const uint16_t *k_pool, *v_pool;
  uint16_t *k_out, *v_out;        // [Hkv][n][D]
  const int32_t *table;
  int32_t layer, begin, n, n_kv_heads, head_dim, page_size;
  uint32_t n_pages;
};
cudaError_t launch_task_read(const ReadParams &p, cudaStream_t stream);

// ---------------------------------------------------------------------------------------------
// S5 / S6: patch attention
// ---------------------------------------------------------------------------------------------
struct AttnTaskDev {     // 32 B, one per task of a (batched) patch call
  int32_t table_off;     // int32 index of the task's page table inside the table region
  int32_t n;             // patch tokens of this task
  int32_t tok_off;       // first row of this task in q/k/v/out/positions
  int32_t kv_len;        // positions[n-1] + 1
  int32_t n_splits;      // KV splits for this task (<= max_splits)
  int32_t split_len;     // tokens per split, multiple of the KV tile
  int32_t pad0, pad1;
};

struct AttnParams {
  const uint16_t *q;         // [n_layers][n_total][Hq][D]
  uint16_t *out;             // same shape
  const uint16_t *k_pool, *v_pool;
  const int32_t *tables;
  const int32_t *positions;  // [n_total]
  const AttnTaskDev *tasks;
  const int32_t *tok_splits; // [n_total] n_splits of the token's task (combine kernel)
  float *part_o;             // [n_layers][max_splits][n_total][Hq][D]   unnormalised
  float *part_ml;            // [n_layers][max_splits][n_total][Hq][2]   (m in log2 units, l)
  int32_t n_total, n_layers, layer_begin, n_q_heads, n_kv_heads, group, page_size, n_tasks;
  int32_t max_splits, max_row_groups;
  uint32_t n_pages;
  float scale_log2;          // log2(e) / sqrt(D)
  const int4 *items;         // mixed-class launch: {class, task index, row group, split} per work item (else NULL)
  int32_t n_items;
  int32_t head_dim;          // the real head_dim (q / out / partial row length); the tcgen05 kernels may run at a padded width
};

// split-KV warp-MMA (mma.sync m16n8k16) path; rows_per_cta in {16, 32, 64}
cudaError_t launch_attn_split(const AttnParams &p, int head_dim, int rows_per_cta, cudaStream_t stream);
cudaError_t launch_attn_combine(const AttnParams &p, int head_dim, cudaStream_t stream);
int attn_split_ctas_per_sm(int head_dim);

// A TMA tensor map (CUtensorMap: 128 opaque bytes, 64-byte aligned), kept free of <cuda.h> here.
struct alignas(64) TmaDesc {
  unsigned char bytes[128];
};

// tcgen05 / TMEM path; q_tiles = 128-row Q tiles per CTA (1 or 2), p.max_row_groups counts groups of
// q_tiles*128 rows.  tm_k / tm_v describe the K / V pool as a 5-D bf16 tensor (D, P, Hkv, n_pages, L)
// with box (64, P, 1, 1, 1) and 128B swizzle (make_pool_tensor_map).
cudaError_t launch_attn_tc(const AttnParams &p, int head_dim, int q_tiles, int parity_streams, const TmaDesc *tm_k,
                           const TmaDesc *tm_v, cudaStream_t stream);
int attn_tc_ctas_per_sm(int head_dim, int q_tiles, int parity_streams);
cudaError_t launch_attn_tc_mixed(const AttnParams &p, const TmaDesc *tm_k, const TmaDesc *tm_v, cudaStream_t stream);
// CTA-pair variant (tcgen05 cta_group::2, clusters of 2) for the > 128-rows class at head_dim 128; same parameters,
// p.max_row_groups counts groups of 256 rows (fcg_attn_pair.cu)
cudaError_t launch_attn_pair(const AttnParams &p, const TmaDesc *tm_k, const TmaDesc *tm_v, cudaStream_t stream);

}  // namespace fcg
