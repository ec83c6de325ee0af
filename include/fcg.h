/* fcg.h -- C ABI of the B200-native FCGRAFT KV-cache grafting library (libfcg.so).
 *
 * What the calls compute is defined by the paper (PAPER.md = the text of arxiv/paper_2606_13097)
 * and, where the paper is silent, by the readings R1..R29 in DESIGN.md:
 *
 *   segment library   the KV half of the two-tier code cache H = (I, C), Eq. (2), PAPER.md:66-79:
 *                     per function a cached K/V state that can be re-injected "without being tied
 *                     to fixed prefix positions".
 *   cache-stitching   Eq. (4): cached KV states are "concatenated and
 *                     injected ... as additional context", each module "preserving its internal
 *                     token order during composition".  Keys are re-rotated by the
 *                     integer position delta (RoPE group law, R1), values are bit-copied.
 *   cache-patching    Eq. (6): the prefix KV is reused, only the middle span
 *                     is recomputed; its fresh K/V are scattered into the cache and the patch
 *                     queries attend causally over the stitched cache (R12).
 *
 * Conventions
 *   - Plain C, no exceptions cross the boundary.  Every call returns an fcg_status_t; on a non-OK
 *     status fcg_last_error() (thread-local, R28) holds a message and the library state is unchanged:
 *     every host-side check of a call happens before any allocation, copy or launch
 *     (allocate-then-commit).  FCG_ERR_CUDA is the exception: a CUDA runtime failure in the middle of a
 *     call may leave work enqueued.
 *   - "device" pointers are CUDA device pointers valid on the library's device; "host" pointers are
 *     ordinary host memory read only during the call (unless stated otherwise).  Every call makes the
 *     library's device current for its own duration and puts the caller's current device back.
 *   - All device work is enqueued on the given `stream` (a cudaStream_t passed as void*; NULL = the
 *     legacy default stream).  Calls return after enqueueing.  Calls on one library must come from
 *     one thread at a time.  Streams (R29): the scratch area, the plan blobs and recycled pages are
 *     library-wide, so a call issued on another stream than the previous call on this library first
 *     waits (one event) for that call's device work; consecutive calls on one stream pay nothing.
 *     The exception is fcg_segment_release, which enqueues nothing (see there), and calls made while
 *     the stream is being captured into a CUDA graph (only fcg_patch_planned may be: see there).
 *   - bf16 everywhere for K, V, q, out (2 bytes/element, the bit layout of __nv_bfloat16).
 *   - The library owns everything inside `arena` (page pool, page tables, segments, workspace); the
 *     caller owns the arena allocation itself and all q/k/v/out buffers.
 *   - There is no CPU fallback and no other backend: without a CUDA device every compute call fails
 *     with FCG_ERR_CUDA.
 */
#ifndef FCG_H_
#define FCG_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct fcg_library fcg_library_t; /* opaque */
typedef int32_t fcg_status_t;

enum {
  FCG_OK = 0,
  FCG_ERR_INVALID_ARG = -1,  /* null pointer, bad geometry, bad shape, positions not increasing */
  FCG_ERR_BAD_SEGMENT = -2,  /* unknown / released segment id */
  FCG_ERR_RANGE = -3,        /* source or destination token range out of bounds */
  FCG_ERR_OVERLAP = -4,      /* plan entries / holes overlap */
  FCG_ERR_UNFILLED = -5,     /* a patch query would attend over a position nobody has filled */
  FCG_ERR_OUT_OF_PAGES = -6, /* page pool (or per-task page-table stride) exhausted */
  FCG_ERR_OUT_OF_ARENA = -7, /* arena / segment table / workspace too small */
  FCG_ERR_CUDA = -8,         /* a CUDA runtime call failed; message has the CUDA error string */
  FCG_ERR_BAD_TASK = -9      /* task id out of range, already live (stitch) or not live (patch) */
};

enum { FCG_ROPE_NONE = 0, FCG_ROPE_HALF_SPLIT = 1, FCG_ROPE_INTERLEAVED = 2 };
enum { FCG_STORE_BF16 = 0, FCG_STORE_FP8_E4M3 = 1 };   /* storage format of a library segment */

/* Geometry and capacities, fixed at create time.
 * Arena layout (all offsets 256-byte aligned, reported by fcg_pool_info):
 *   K pool  [n_layers][n_pages][n_kv_heads][page_size][head_dim] bf16   ("HND" pages: one head's
 *   V pool  same shape                                                   slice of a page is contiguous)
 *   page tables  int32 [max_tasks][ceil(max_task_tokens / page_size)]
 *   workspace    workspace_bytes (split-KV partials, host-call staging, plan blobs)
 *   segments     the rest, first-fit; a segment is K [n_layers][n_kv_heads][n][head_dim] then V. */
typedef struct {
  int32_t n_layers;
  int32_t n_q_heads;       /* multiple of n_kv_heads */
  int32_t n_kv_heads;
  int32_t head_dim;        /* a multiple of 16 in [16, 256] (R27).  64, 128 and 256 have kernels of their own; the others run
                              the gather with head_dim as a run-time value and the tcgen05 attention at the next of those
                              widths with zero-padded columns.  Only 64 and 128 also have the split-KV warp-MMA kernel */
  int32_t page_size;       /* tokens per page: 8, 16, 32 or 64 */
  int32_t rope_mode;       /* FCG_ROPE_NONE: stitch is a pure gather; FCG_ROPE_HALF_SPLIT: pairs (j, j + head_dim/2) (R2);
                              FCG_ROPE_INTERLEAVED: pairs (2j, 2j + 1) */
  double rope_base;        /* theta_j = rope_base^(-2j/head_dim) (R3); ignored if inv_freq != NULL */
  const double *inv_freq;  /* host, optional [head_dim/2] override (scaled RoPE); copied at create */
  void *arena;             /* device */
  uint64_t arena_bytes;
  int32_t max_segments;
  int32_t max_tasks;
  int32_t max_task_tokens; /* largest length a single task may reach (sizes the per-task page table); a task may grow up
                              to it by appending patches (R25) */
  uint32_t n_pages;        /* pages in the pool, shared by all live tasks */
  uint64_t workspace_bytes;/* 0 -> 256 MiB */
  int32_t device;          /* CUDA device ordinal the arena lives on */
  void *host_arena;        /* optional second tier (Eq. 3): PINNED host memory (cudaHostAlloc / cudaHostRegister, e.g. a
                              torch pin_memory tensor), 256-byte aligned, caller-owned; NULL -> no host tier */
  uint64_t host_arena_bytes;
} fcg_config_t;

/* Bytes of arena needed for a configuration that must hold `segment_tokens` library tokens in total
 * (host-only arithmetic, works without a GPU).  Returns 0 on a bad configuration. */
uint64_t fcg_arena_bytes_required(const fcg_config_t *cfg, uint64_t segment_tokens);

/* Creates a library over cfg->arena.  Fails with INVALID_ARG (geometry), OUT_OF_ARENA (arena too small
 * for pool + tables + workspace) or CUDA. */
fcg_status_t fcg_library_create(const fcg_config_t *cfg, fcg_library_t **out);
/* Synchronises the device, then frees host state.  The arena is the caller's. */
fcg_status_t fcg_library_destroy(fcg_library_t *lib);

/* S1 (Eq. 2).  Copies n_tokens of K and V into the library.  k, v: device bf16, logical shape
 * [n_layers][n_kv_heads][n_tokens][head_dim]; strides in ELEMENTS for those four axes (NULL =
 * contiguous; strides[3] must be 1).  orig_start >= 0 is the position at which token 0's key was
 * RoPE-encoded.  The caller may free k/v once `stream` has passed this call.  The id returned is the
 * smallest id not in use. */
fcg_status_t fcg_segment_register(fcg_library_t *lib, const void *k, const void *v, int32_t n_tokens,
                                  int32_t orig_start, const int64_t *strides, void *stream,
                                  int32_t *seg_id_out);
/* S1 with fp8 storage (memory pressure of the code cache: PAPER.md:81-87; R26).
 * Same arguments as fcg_segment_register; the bf16 rows are quantised once, here: every stored row (the head_dim
 * elements of one (layer, kv head, token)) keeps OCP E4M3 codes (1 byte per element) and one power-of-two scale
 * 2^e (1 byte, e + 127): e = the smallest integer with max|x| <= 448 * 2^e over the row's finite elements, clamped
 * to [-127, 127], 0 for an all-zero row; code = RNE_e4m3(x * 2^-e); +-inf and NaN have no E4M3 value and become the
 * NaN code.  The segment takes (head_dim + 1) / (2 head_dim) of the bf16 bytes.  Plans, offload / prefetch and
 * release treat it like any segment; fcg_stitch de-quantises (exactly) BEFORE the rotation, so a shifted key is one
 * rounding away from the exact rotation of the stored value, and values are the de-quantised values rounded to
 * bf16 (exact outside bf16's subnormal range).  The paged cache itself stays bf16. */
fcg_status_t fcg_segment_register_fp8(fcg_library_t *lib, const void *k, const void *v, int32_t n_tokens,
                                      int32_t orig_start, const int64_t *strides, void *stream, int32_t *seg_id_out);
/* Storage format (FCG_STORE_*) and bytes a segment occupies in its tier; either output may be NULL. */
fcg_status_t fcg_segment_storage(fcg_library_t *lib, int32_t seg_id, int32_t *format, uint64_t *bytes);
/* Copies the stored representation of a segment out (tests, inspection): k_out, v_out [n_layers][n_kv_heads][n][head_dim]
 * -- bf16, or uint8 E4M3 codes for an fp8 segment, whose scale bytes (e + 127) go to k_exp_out, v_exp_out
 * [n_layers][n_kv_heads][n] (required then, ignored otherwise).  Device or host destinations.  Asynchronous on `stream`. */
fcg_status_t fcg_segment_read(fcg_library_t *lib, int32_t seg_id, void *k_out, void *v_out, void *k_exp_out,
                              void *v_exp_out, void *stream);
/* The caller guarantees no enqueued stitch still reads the segment. */
fcg_status_t fcg_segment_release(fcg_library_t *lib, int32_t seg_id);

typedef struct { int32_t seg_id, src_begin, n_tokens, dst_offset; } fcg_plan_entry_t;
typedef struct { int32_t begin, n_tokens; } fcg_hole_t;            /* ranges left for patches */
typedef struct {
  int32_t task_id;                  /* chosen by the caller in [0, max_tasks); must not be live */
  const fcg_plan_entry_t *entries;  /* host */
  int32_t n_entries;
  const fcg_hole_t *holes;          /* host; may be NULL if n_holes == 0 */
  int32_t n_holes;
  int32_t capacity_tokens;          /* 0 -> max end of entries/holes; pages are reserved for the capacity.  A reservation,
                                       not a limit: later patches may append beyond it (R25) */
} fcg_plan_t;

/* S2 + S3 (Eq. 4).  For every plan: validates it (R5-R7: 0 <= src_begin, n > 0, src_begin + n <= n_seg,
 * dst_offset >= 0, end <= capacity <= max_task_tokens; entries and holes pairwise disjoint), computes
 * delta_e = dst_offset - orig_start - src_begin, reserves ceil(capacity / page_size) pages (plans in
 * array order, pages in ascending logical order, from a LIFO pool that initially hands out 0, 1, 2, ...;
 * R9), writes the page table, and launches ONE fused kernel over all plans:
 *     K_out[dst + i][j]       = bf16(a cos(delta theta_j) - b sin(delta theta_j))
 *     K_out[dst + i][j + D/2] = bf16(b cos(delta theta_j) + a sin(delta theta_j)),  (a, b) = K_seg[src + i][j, j + D/2]
 *     V_out[dst + i] = V_seg[src + i]   (bits)
 * Entries with delta 0 (and rope_mode NONE) are bit copies.  Any failing plan fails the whole batch
 * with nothing changed.  Unused tail slots of the last page are never written nor read (R10). */
fcg_status_t fcg_stitch(fcg_library_t *lib, const fcg_plan_t *plans, int32_t n_plans, void *stream);

/* fcg_stitch with overlapped prefetch (Table 19: CPU -> GPU reloads "only
 * when a required function cache is not resident").  Same arguments, same result, same page tables.  Segments of
 * the host tier that the plans name are first copied back to the device tier -- one host->device copy each, on a
 * stream of the library's own, into a first-fit arena range (a segment that finds no room stays offloaded and is read
 * in place, as fcg_stitch does) -- WHILE the entries of the resident segments are being stitched on `stream`; the
 * entries of the prefetched segments are stitched by a second launch on `stream` once their copies have landed.  On
 * return (status OK) those segments are resident, as after fcg_segment_prefetch. */
fcg_status_t fcg_stitch_prefetch(fcg_library_t *lib, const fcg_plan_t *plans, int32_t n_plans, void *stream);

/* S4 + S5/S6 (Eq. 6).  q [n_layers][n][n_q_heads][head_dim], k, v [n_layers][n][n_kv_heads][head_dim],
 * out [n_layers][n][n_q_heads][head_dim]: device bf16, contiguous, for cache layers
 * [layer_begin, layer_begin + n_layers).  k (and q) are already position-encoded by the caller (R13).
 * positions: host int32[n], strictly increasing, in [0, max_task_tokens).  Positions at or beyond the task's
 * capacity APPEND (R25): the task grows to positions[n-1] + 1 and takes the missing pages from the
 * pool at the time of the call (ascending logical order, tasks of a batch in array order; OUT_OF_PAGES leaves
 * everything unchanged) -- so a caller can decode the x_mid of Eq. 6 token by token without knowing its length.
 * For each layer the n fresh K/V rows are
 * written to the slots of `positions` (bit copy), then for each patch token i and q-head h
 *     out[i][h] = softmax_{x <= positions[i]}(q[i][h] . K[x][h / G] / sqrt(head_dim)) V[x][h / G],   G = n_q_heads / n_kv_heads
 * with fp32 softmax/accumulation, bf16 result.  Every x <= positions[n-1] must be filled (stitched, or
 * patched by this or an earlier call), else UNFILLED (a gap between the old end and an appended position is a hole,
 * not an append).  The kernel is chosen by fcg_set_attn_policy (default: tcgen05 / TMEM tiles whenever the geometry
 * has them, the split-KV warp-MMA kernel otherwise).  Not capturable into a CUDA graph (the call uploads a plan blob
 * from pinned host memory): see fcg_patch_plan_create. */
fcg_status_t fcg_patch(fcg_library_t *lib, int32_t task_id, int32_t layer_begin, int32_t n_layers,
                       const void *q, const void *k, const void *v, const int32_t *positions, int32_t n,
                       void *out, void *stream);

/* fcg_patch for callers that hold q and k BEFORE position encoding (R13 variant): token
 * i's q and k rows are first rotated to the absolute position positions[i] with the library's RoPE (theta_j and pair
 * layout of the configuration; each rounded once to bf16, within 1 ulp of the fp64 value), then scattered and attended
 * exactly as in fcg_patch.  FCG_ROPE_NONE: identical to fcg_patch.  The rotated copies live in the workspace
 * (OUT_OF_ARENA if they, or the n x head_dim/2 cos/sin table, do not fit). */
fcg_status_t fcg_patch_rope(fcg_library_t *lib, int32_t task_id, int32_t layer_begin, int32_t n_layers,
                            const void *q, const void *k, const void *v, const int32_t *positions, int32_t n,
                            void *out, void *stream);

/* Same as fcg_patch with q, k, v, out in HOST memory (pinned for true asynchrony): the call enqueues the
 * host->device copies, the kernels and the device->host copy of `out`; out is valid (and q, k, v may be reused)
 * once `stream` has been synchronised.  The host->device copies run on a stream of the library's own, ordered
 * after the previous patch call and joined into `stream` before the kernels, so they overlap whatever else the
 * caller has enqueued on `stream` just before (typically the fcg_stitch of the same graft); calls of 8 MiB of q or
 * more are pipelined in four layer groups (copy in, attend, copy out overlap; the plan blob is uploaded ahead of
 * the big copies on the copy stream, so the first group's kernels do not queue behind them).  Staging comes from the workspace
 * (OUT_OF_ARENA if it does not fit). */
fcg_status_t fcg_patch_host(fcg_library_t *lib, int32_t task_id, int32_t layer_begin, int32_t n_layers,
                            const void *q, const void *k, const void *v, const int32_t *positions, int32_t n,
                            void *out, void *stream);

/* Batched patching (independent tasks, one launch): task_ids host int32[n_tasks] (distinct, live);
 * n_per_task host int32[n_tasks]; positions host int32[sum n], the tasks' position lists back to back;
 * q/k/v/out device bf16 [n_layers][sum n][heads][head_dim].  n_layers * n_tasks <= 65535 per call (the attention grid
 * runs (layer, task) along z; INVALID_ARG otherwise: patch fewer layers or tasks per call). */
fcg_status_t fcg_patch_batch(fcg_library_t *lib, const int32_t *task_ids, const int32_t *n_per_task,
                             int32_t n_tasks, int32_t layer_begin, int32_t n_layers, const void *q,
                             const void *k, const void *v, const int32_t *positions, void *out, void *stream);

/* fcg_patch_batch with q, k, v, out in HOST memory: staging, copy streams and layer-group pipelining as fcg_patch_host. */
fcg_status_t fcg_patch_batch_host(fcg_library_t *lib, const int32_t *task_ids, const int32_t *n_per_task,
                                  int32_t n_tasks, int32_t layer_begin, int32_t n_layers, const void *q,
                                  const void *k, const void *v, const int32_t *positions, void *out, void *stream);

/* Patch plans: the per-layer call pattern of a real model without per-call host work, and CUDA-graph capture.
 * fcg_patch_plan_create does everything of fcg_patch_batch that does not depend on the tensors -- validation (R6),
 * growth (R25), split selection for `layers_per_call` layers on the GPU at a time (the layers of one call, or -- for
 * per-layer calls forked over several streams -- the number of calls in flight), the upload of positions / descriptors into a
 * device range of the plan's own (taken from the segment arena; OUT_OF_ARENA), and the COMMIT of the fill state:
 * the positions count as filled from here on, the caller runs the plan for every layer before relying on them.
 * fcg_patch_planned then only launches scatter -> attention (-> combine) for layers [layer_begin, layer_begin +
 * n_layers) with q, k, v, out as in fcg_patch_batch; it may be called any number of times, with any tensors, and
 * may be captured into a CUDA graph (it makes no copies and touches no host state besides launch statistics; while
 * the stream is capturing, the stream-ordering rule above is skipped and the caller orders the graph against other
 * work on the library).  Planned calls for DISJOINT layer ranges touch disjoint memory (their split-KV partials live
 * in per-layer slots in the lower half of the workspace's scratch area -- the upper half is where the host variants
 * stage; OUT_OF_ARENA at plan creation if the slots do not fit there), so inside a capture they
 * may be forked over several streams and run concurrently.  BAD_TASK if a task of the plan was released,
 * re-stitched or moved by fcg_task_shift since (a shift un-fills positions and re-assigns pages: make a new plan).
 * Destroy returns the device range to the segment arena with no stream ordering: the caller guarantees no enqueued work
 * still reads it, and a CUDA graph captured from the plan must be destroyed (or never replayed again) BEFORE the plan
 * is -- a replay after that reads whatever segment was registered into the range next.  Destroying a plan twice is
 * INVALID_ARG.  fcg_library_destroy frees the plans the caller did not destroy. */
typedef struct fcg_patch_plan fcg_patch_plan_t;
fcg_status_t fcg_patch_plan_create(fcg_library_t *lib, const int32_t *task_ids, const int32_t *n_per_task, int32_t n_tasks,
                                   const int32_t *positions, int32_t layers_per_call, void *stream, fcg_patch_plan_t **out);
fcg_status_t fcg_patch_planned(fcg_library_t *lib, fcg_patch_plan_t *plan, int32_t layer_begin, int32_t n_layers,
                               const void *q, const void *k, const void *v, void *out, void *stream);
fcg_status_t fcg_patch_plan_destroy(fcg_library_t *lib, fcg_patch_plan_t *plan);

/* Device pointer to the task's page table (int32[n_pages], logical page -> physical page id), its page
 * count and current token count T (max end of stitched/declared/patched ranges).  Token x lives at
 * (table[x / page_size], x % page_size). */
fcg_status_t fcg_task_page_table(fcg_library_t *lib, int32_t task_id, const int32_t **dev_table,
                                 int32_t *n_pages, int32_t *n_tokens);
/* Host copy of the same table (no device access): writes min(n_pages, cap) entries to `out`. */
fcg_status_t fcg_task_page_table_host(fcg_library_t *lib, int32_t task_id, int32_t *out, int32_t cap,
                                      int32_t *n_pages);
/* Boundary-recompute plan (the related work of PAPER.md:47, 588): the positions worth
 * recomputing after a stitch -- the first `width` tokens of every stitched entry that does not start at position 0,
 * ascending and without duplicates.  Host only.  Writes min(count, cap) positions to `out` (may be NULL with cap 0)
 * and the count to *n_out; the caller recomputes those tokens with the model and hands them to fcg_patch (re-patching
 * a filled position overwrites it, R14).  Describes the stitch; later fcg_task_shift moves are not tracked. */
fcg_status_t fcg_task_boundary_positions(fcg_library_t *lib, int32_t task_id, int32_t width, int32_t *out, int32_t cap,
                                         int32_t *n_out);
/* Returns the task's pages to the pool (pushed so that they are re-issued in ascending logical order).  Enqueues
 * nothing: work still in flight on the task is protected by the stream rule above (the next call that could reuse
 * the pages on another stream waits for it). */
fcg_status_t fcg_task_release(fcg_library_t *lib, int32_t task_id);

/* Two-tier residency (Eq. 3; transfer cost in Table 19).
 * Which entries to move is the caller's policy (the locality score is not on the path); the library moves bits.
 * fcg_segment_offload: device -> host tier (one async copy on `stream`), the arena range is returned to the
 *   segment allocator.  fcg_segment_prefetch: host tier -> device (first-fit arena range, one async copy), the host
 *   range is returned.  Both are no-ops when the segment already is where it is asked to be.  INVALID_ARG without a
 *   host tier, BAD_SEGMENT, OUT_OF_ARENA when the receiving tier has no free range (state unchanged).
 * A plan may name an offloaded segment: fcg_stitch then reads it straight from the pinned host range (zero-copy
 *   over the host link), with the same result.  fcg_segment_release frees whichever tier holds the segment.
 * fcg_segment_info: any of the three outputs may be NULL; resident = 1 (device) or 0 (host tier). */
fcg_status_t fcg_segment_offload(fcg_library_t *lib, int32_t seg_id, void *stream);
fcg_status_t fcg_segment_prefetch(fcg_library_t *lib, int32_t seg_id, void *stream);
fcg_status_t fcg_segment_info(fcg_library_t *lib, int32_t seg_id, int32_t *n_tokens, int32_t *orig_start,
                              int32_t *resident);

/* Suffix re-graft of a length-changing patch (Eq. 6, R15):
 * moves cache positions [src_begin, src_begin + n_tokens) of a live task to [dst_begin, dst_begin + n_tokens),
 * all layers and kv heads: keys re-rotated by delta = dst_begin - src_begin (the stitch rule R1; bit copy for
 * FCG_ROPE_NONE), values bit-copied.  Source positions become unfilled, destination positions filled (filled
 * destination positions are overwritten); T never shrinks.  The source must lie inside the task's capacity and the
 * destination inside [0, max_task_tokens) (RANGE); a destination beyond the capacity grows the task like an appending
 * patch (R25: gap pages, then destination pages, ascending).  Every source position must be filled (UNFILLED).  The ranges may overlap: every logical page the
 * destination touches is given a fresh page from the pool (ascending logical order; OUT_OF_PAGES if the pool
 * cannot supply them), slots of those pages outside the destination keep their contents, and the replaced pages
 * return to the pool by the rule of fcg_task_release -- so the task's page table changes.  delta == 0 is a
 * no-op.  Asynchronous on `stream`; a failing call leaves the library unchanged. */
fcg_status_t fcg_task_shift(fcg_library_t *lib, int32_t task_id, int32_t src_begin, int32_t n_tokens,
                            int32_t dst_begin, void *stream);

/* Segment extraction (`update` of Alg. 1B): cuts cache positions
 * [begin, begin + n_tokens) of a live task, all layers and kv heads, into a new library segment without a host
 * round trip.  Keys are re-rotated by delta = new_orig_start - begin, i.e. stored as if the segment's first
 * token sat at position new_orig_start (begin: bit copy; 0: canonical form); values are bit-copied.  The range
 * must lie inside the capacity (RANGE) and be filled (UNFILLED); new_orig_start >= 0.  The id is the lowest free
 * one, as for fcg_segment_register; OUT_OF_ARENA as there.  Asynchronous on `stream`. */
fcg_status_t fcg_segment_extract(fcg_library_t *lib, int32_t task_id, int32_t begin, int32_t n_tokens,
                                 int32_t new_orig_start, void *stream, int32_t *seg_id_out);

/* Gathers logical tokens [begin, begin + n) of one layer of a task's cache into contiguous device
 * buffers k_out, v_out [n_kv_heads][n][head_dim] (bit copy through the page table; for tests and for
 * callers that need a dense view). */
fcg_status_t fcg_task_read(fcg_library_t *lib, int32_t task_id, int32_t layer, int32_t begin, int32_t n,
                           void *k_out, void *v_out, void *stream);

typedef struct {
  uint64_t k_pool_offset, v_pool_offset;  /* byte offsets into the arena */
  uint64_t pool_bytes;                    /* bytes of ONE pool */
  uint64_t page_table_offset, workspace_offset, segments_offset;
  uint64_t segments_bytes_free;
  uint32_t n_pages, n_pages_free;
  int32_t n_segments_live, n_tasks_live;
} fcg_pool_info_t;
fcg_status_t fcg_pool_info(fcg_library_t *lib, fcg_pool_info_t *out);

/* Kernel selection for patch attention: calls whose largest task has R = n * G >= tc_min_rows query rows per
 * kv head use the tcgen05/TMEM kernel, others the split-KV warp-MMA kernel.  Default 1: tcgen05 for every R
 * (measured faster than the split-KV kernel down to a decode step, DESIGN.md section 6 -- north_star expected the
 * opposite for short patches); INT32_MAX = never.  Every head_dim other than 64 and 128 always runs the tcgen05 kernel (no
 * split-KV warp-MMA instantiation): tc_min_rows is ignored there, force_splits applies.
 * force_splits > 0 fixes the number of KV splits per task (clamped to the task's 64-token tile count);
 * 0 = the library's wave-filling choice.  The result does not depend on either knob beyond summation order
 * (P11, split invariance). */
fcg_status_t fcg_set_attn_policy(fcg_library_t *lib, int32_t tc_min_rows, int32_t force_splits);
/* Tasks with more than 128 query rows per kv head (head_dim 128) run on single CTAs holding two Q tiles (default,
 * enable == 0) or on CTA pairs -- clusters of two CTAs sharing every K / V tile through tcgen05 cta_group::2
 * (enable != 0; measured: equal on the power-capped C5, 10-15 % slower on C3 / C4).  Same
 * results up to summation order. */
fcg_status_t fcg_set_attn_pairs(fcg_library_t *lib, int32_t enable);
/* A batch whose tasks fall into several CTA classes (<= 64, 65..128, > 128 query rows per kv head; head_dim 128) runs as
 * one launch per class, longest class first (default, enable == 0), or as ONE launch with the classes interleaved
 * (enable != 0; measured equal on C4: the classes do not speed each other up). */
fcg_status_t fcg_set_attn_mixed(fcg_library_t *lib, int32_t enable);

/* Launch statistics since create (kernels launched by this library; bench.py reports them). */
typedef struct {
  uint64_t stitch_launches, register_launches, scatter_launches, attn_split_launches, attn_combine_launches,
      attn_tc_launches, read_launches;
  int32_t last_attn_path;   /* 0 none, 1 split-KV warp-MMA, 2 tcgen05 */
  int32_t last_attn_splits;
  uint64_t offload_copies, prefetch_copies;   /* tier moves (copy engine, not kernels) */
  uint64_t rope_qk_launches;
} fcg_stats_t;
fcg_status_t fcg_stats(fcg_library_t *lib, fcg_stats_t *out);

/* Locality score of the cache management scheme (Eq. 3, 8, 9, 10): host-only bookkeeping, no
 * CUDA, independent of any library handle.  Ids are the caller's function ids (normally segment ids).
 *   l(f_k) = (1 - l_curr) (alpha l_freq + beta sum_j l_asso(f_j | f_k) + gamma l_sema) + l_curr
 *   l_freq = count(f_k) / max_j count(f_j);  l_asso(f_j | f_k) = cooccur(f_k, f_j) / count(f_k);  l_sema = PPL / max PPL.
 * Readings (R24): fcg_scorer_record takes ONE task's execution trace, the functions in invocation order;
 * count = invocations over all recorded traces; cooccur(f_k, f_j) = times f_j was the next invocation after f_k (j != k),
 * so the sum over j lies in [0, 1]; l_curr = 1 for the functions of the most recent trace; PPL comes from the caller
 * (0 where never set).  fcg_scorer_rank sorts `ids` by ascending score (ties: ascending id): the front of the list is
 * what to hand to fcg_segment_offload first.  fcg_scorer_forget drops a released function from the statistics. */
typedef struct fcg_scorer fcg_scorer_t;
fcg_status_t fcg_scorer_create(fcg_scorer_t **out);
fcg_status_t fcg_scorer_destroy(fcg_scorer_t *s);
fcg_status_t fcg_scorer_record(fcg_scorer_t *s, const int32_t *ids, int32_t n);
fcg_status_t fcg_scorer_set_ppl(fcg_scorer_t *s, int32_t id, double ppl);
fcg_status_t fcg_scorer_forget(fcg_scorer_t *s, int32_t id);
fcg_status_t fcg_scorer_score(fcg_scorer_t *s, int32_t id, double alpha, double beta, double gamma, double *score);
fcg_status_t fcg_scorer_rank(fcg_scorer_t *s, const int32_t *ids, int32_t n, double alpha, double beta, double gamma,
                             int32_t *ids_out, double *scores_out);

/* The key re-rotation of cache-stitching (Eq. 4; RoPE group law, R1) for callers that are not
 * allowed to allocate device memory.
 *
 * Who that is: a plug-in inside a serving engine that claimed all of HBM for its own block pool at start-up (a
 * cudaMalloc there fails, or takes memory the engine believes it owns); code that runs while another thread of the
 * process records a CUDA graph in global capture mode (the runtime refuses cudaMalloc for everybody until the capture
 * ends); and latency-critical loops that cannot afford the device-wide synchronisation an allocation or a free may
 * bring.  Such callers also cannot build an fcg_library_t just for one segment, because a library needs an arena with
 * a workspace.  This call needs neither: it allocates nothing, on the host or on the device, and uses no handle.
 *
 * What it does: reads one dense bf16 segment  k_src, v_src  [n_layers][n_kv_heads][n_tokens][head_dim]  and writes
 * k_dst, v_dst of the same shape: every key rotated by the angle  delta * theta_j  (theta_j = inv_freq[j] when
 * inv_freq is given -- head_dim / 2 host doubles read during the call -- else rope_base^(-2j / head_dim)), every
 * value copied bit for bit.  delta == 0 or FCG_ROPE_NONE copies the keys too.  It is the same kernel with the same
 * arithmetic as fcg_stitch, so the bits equal those of stitching the segment at distance delta from where it was
 * encoded.  All four buffers are device memory of the CURRENT device (there is no library whose device could be
 * made current), 16-byte aligned, owned by the caller; no destination may overlap a source or the other
 * destination (OVERLAP).  head_dim: a multiple of 16 in [16, 256]; n_layers <= 65535; n_tokens == 0 is a no-op.
 *
 * Where the scratch lives: the kernel reads a small plan (entry descriptor, chunk list, the cos / sin table of
 * delta).  For this call the plan sits in a fixed 67 840-byte array inside the library image, present on every GPU
 * that loads libfcg.so for as long as the process lives.  Its size is what bounds a call:
 * n_tokens <= FCG_STATIC_SHIFT_MAX_TOKENS (also returned by fcg_segment_shift_static_max_tokens); a longer segment
 * is refused with FCG_ERR_RANGE and a message that names the limit -- split it into several calls, or use a library.
 *
 * Sharing: there is ONE such array per GPU, and each call first overwrites the part of it that it is going to read
 * (nothing needs to be zero, nothing of an earlier call is relied upon).  Two calls are therefore only safe when
 * the GPU runs them one after the other: same stream, or streams ordered by an event.  Calls that may overlap on
 * the device race on the plan and produce garbage in both destinations; the library does not detect that.
 *
 * First call on a device: it looks up the device address of the array (one runtime query, cached per device
 * ordinal, thread-safe).  Make that first call during start-up, outside any stream capture.
 *
 * Asynchronous on `stream`: two kernel launches, no copy.  Errors: INVALID_ARG (shape, alignment, NULL, rope
 * parameters), RANGE (too many tokens), OVERLAP, CUDA.  Every check happens before anything is enqueued. */
#define FCG_STATIC_SHIFT_MAX_TOKENS 65536
fcg_status_t fcg_segment_shift_static(const void *k_src, const void *v_src, void *k_dst, void *v_dst, int32_t n_layers,
                                      int32_t n_kv_heads, int32_t n_tokens, int32_t head_dim, int32_t rope_mode,
                                      double rope_base, const double *inv_freq, int32_t delta, void *stream);
int32_t fcg_segment_shift_static_max_tokens(void);

/* Message for the last non-OK status returned on this thread (never NULL). */
const char *fcg_last_error(void);
/* "x.y.z sm_100a" */
const char *fcg_version(void);

#ifdef __cplusplus
}
#endif
#endif /* FCG_H_ */
