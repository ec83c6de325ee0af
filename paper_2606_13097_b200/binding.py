"""ctypes binding of libfcg.so (include/fcg.h).  Argument marshalling only: every step of the hot
path (gather + RoPE shift, scatter, patch attention) runs in the CUDA kernels behind the C ABI.

The functions ``fcg_*`` mirror the C entry points one to one and take raw pointers / ints (or torch
tensors, whose ``data_ptr()`` is passed).  ``FcgLibrary`` is a small convenience wrapper over them.
PyTorch is used for device memory and streams only.  There is no CPU fallback: if libfcg.so has not
been built, importing works but the first call raises ``FcgError`` telling how to build it.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
# FCG_LIBRARY: another build of the same library (the ASan / UBSan build of `python -m paper_2606_13097_b200.build --sanitize`)
LIB_PATH = os.environ.get("FCG_LIBRARY") or os.path.join(_HERE, "libfcg.so")

FCG_OK = 0
FCG_ERR_INVALID_ARG = -1
FCG_ERR_BAD_SEGMENT = -2
FCG_ERR_RANGE = -3
FCG_ERR_OVERLAP = -4
FCG_ERR_UNFILLED = -5
FCG_ERR_OUT_OF_PAGES = -6
FCG_ERR_OUT_OF_ARENA = -7
FCG_ERR_CUDA = -8
FCG_ERR_BAD_TASK = -9

FCG_ROPE_NONE = 0
FCG_ROPE_HALF_SPLIT = 1
FCG_ROPE_INTERLEAVED = 2
FCG_STORE_BF16 = 0
FCG_STORE_FP8_E4M3 = 1


class FcgError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"fcg status {status}: {msg}")
        self.status = status


class fcg_config_t(C.Structure):
    _fields_ = [("n_layers", C.c_int32), ("n_q_heads", C.c_int32), ("n_kv_heads", C.c_int32),
                ("head_dim", C.c_int32), ("page_size", C.c_int32), ("rope_mode", C.c_int32),
                ("rope_base", C.c_double), ("inv_freq", C.POINTER(C.c_double)),
                ("arena", C.c_void_p), ("arena_bytes", C.c_uint64),
                ("max_segments", C.c_int32), ("max_tasks", C.c_int32), ("max_task_tokens", C.c_int32),
                ("n_pages", C.c_uint32), ("workspace_bytes", C.c_uint64), ("device", C.c_int32),
                ("host_arena", C.c_void_p), ("host_arena_bytes", C.c_uint64)]


class fcg_plan_entry_t(C.Structure):
    _fields_ = [("seg_id", C.c_int32), ("src_begin", C.c_int32), ("n_tokens", C.c_int32), ("dst_offset", C.c_int32)]


class fcg_hole_t(C.Structure):
    _fields_ = [("begin", C.c_int32), ("n_tokens", C.c_int32)]


class fcg_plan_t(C.Structure):
    _fields_ = [("task_id", C.c_int32), ("entries", C.POINTER(fcg_plan_entry_t)), ("n_entries", C.c_int32),
                ("holes", C.POINTER(fcg_hole_t)), ("n_holes", C.c_int32), ("capacity_tokens", C.c_int32)]


class fcg_pool_info_t(C.Structure):
    _fields_ = [("k_pool_offset", C.c_uint64), ("v_pool_offset", C.c_uint64), ("pool_bytes", C.c_uint64),
                ("page_table_offset", C.c_uint64), ("workspace_offset", C.c_uint64), ("segments_offset", C.c_uint64),
                ("segments_bytes_free", C.c_uint64), ("n_pages", C.c_uint32), ("n_pages_free", C.c_uint32),
                ("n_segments_live", C.c_int32), ("n_tasks_live", C.c_int32)]


class fcg_stats_t(C.Structure):
    _fields_ = [("stitch_launches", C.c_uint64), ("register_launches", C.c_uint64), ("scatter_launches", C.c_uint64),
                ("attn_split_launches", C.c_uint64), ("attn_combine_launches", C.c_uint64),
                ("attn_tc_launches", C.c_uint64), ("read_launches", C.c_uint64),
                ("last_attn_path", C.c_int32), ("last_attn_splits", C.c_int32),
                ("offload_copies", C.c_uint64), ("prefetch_copies", C.c_uint64), ("rope_qk_launches", C.c_uint64)]


# every symbol include/fcg.h declares: name -> (restype, argtypes)
_P = C.c_void_p
_I = C.c_int32
_PI = C.POINTER(C.c_int32)
SYMBOLS = {
    "fcg_arena_bytes_required": (C.c_uint64, [C.POINTER(fcg_config_t), C.c_uint64]),
    "fcg_library_create": (_I, [C.POINTER(fcg_config_t), C.POINTER(_P)]),
    "fcg_library_destroy": (_I, [_P]),
    "fcg_segment_register": (_I, [_P, _P, _P, _I, _I, C.POINTER(C.c_int64), _P, _PI]),
    "fcg_segment_register_fp8": (_I, [_P, _P, _P, _I, _I, C.POINTER(C.c_int64), _P, _PI]),
    "fcg_segment_storage": (_I, [_P, _I, _PI, C.POINTER(C.c_uint64)]),
    "fcg_segment_read": (_I, [_P, _I, _P, _P, _P, _P, _P]),
    "fcg_segment_release": (_I, [_P, _I]),
    "fcg_segment_offload": (_I, [_P, _I, _P]),
    "fcg_segment_prefetch": (_I, [_P, _I, _P]),
    "fcg_segment_info": (_I, [_P, _I, _PI, _PI, _PI]),
    "fcg_stitch": (_I, [_P, C.POINTER(fcg_plan_t), _I, _P]),
    "fcg_stitch_prefetch": (_I, [_P, C.POINTER(fcg_plan_t), _I, _P]),
    "fcg_patch": (_I, [_P, _I, _I, _I, _P, _P, _P, _PI, _I, _P, _P]),
    "fcg_patch_host": (_I, [_P, _I, _I, _I, _P, _P, _P, _PI, _I, _P, _P]),
    "fcg_patch_rope": (_I, [_P, _I, _I, _I, _P, _P, _P, _PI, _I, _P, _P]),
    "fcg_patch_batch": (_I, [_P, _PI, _PI, _I, _I, _I, _P, _P, _P, _PI, _P, _P]),
    "fcg_patch_batch_host": (_I, [_P, _PI, _PI, _I, _I, _I, _P, _P, _P, _PI, _P, _P]),
    "fcg_patch_plan_create": (_I, [_P, _PI, _PI, _I, _PI, _I, _P, C.POINTER(_P)]),
    "fcg_patch_planned": (_I, [_P, _P, _I, _I, _P, _P, _P, _P, _P]),
    "fcg_patch_plan_destroy": (_I, [_P, _P]),
    "fcg_task_page_table": (_I, [_P, _I, C.POINTER(_P), _PI, _PI]),
    "fcg_task_page_table_host": (_I, [_P, _I, _PI, _I, _PI]),
    "fcg_task_release": (_I, [_P, _I]),
    "fcg_task_boundary_positions": (_I, [_P, _I, _I, _PI, _I, _PI]),
    "fcg_task_shift": (_I, [_P, _I, _I, _I, _I, _P]),
    "fcg_segment_extract": (_I, [_P, _I, _I, _I, _I, _P, _PI]),
    "fcg_task_read": (_I, [_P, _I, _I, _I, _I, _P, _P, _P]),
    "fcg_pool_info": (_I, [_P, C.POINTER(fcg_pool_info_t)]),
    "fcg_set_attn_policy": (_I, [_P, _I, _I]),
    "fcg_set_attn_pairs": (_I, [_P, _I]),
    "fcg_set_attn_mixed": (_I, [_P, _I]),
    "fcg_stats": (_I, [_P, C.POINTER(fcg_stats_t)]),
    "fcg_scorer_create": (_I, [C.POINTER(_P)]),
    "fcg_scorer_destroy": (_I, [_P]),
    "fcg_scorer_record": (_I, [_P, _PI, _I]),
    "fcg_scorer_set_ppl": (_I, [_P, _I, C.c_double]),
    "fcg_scorer_forget": (_I, [_P, _I]),
    "fcg_scorer_score": (_I, [_P, _I, C.c_double, C.c_double, C.c_double, C.POINTER(C.c_double)]),
    "fcg_scorer_rank": (_I, [_P, _PI, _I, C.c_double, C.c_double, C.c_double, _PI, C.POINTER(C.c_double)]),
    "fcg_segment_shift_static": (_I, [_P, _P, _P, _P, _I, _I, _I, _I, _I, C.c_double, C.POINTER(C.c_double), _I, _P]),
    "fcg_segment_shift_static_max_tokens": (_I, []),
    "fcg_last_error": (C.c_char_p, []),
    "fcg_version": (C.c_char_p, []),
}

_lib = None


def load() -> C.CDLL:
    """dlopen libfcg.so (once).  Fails loudly when it has not been built -- there is no fallback."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise FcgError(FCG_ERR_CUDA, f"{LIB_PATH} is missing: build it with "
                                         "`python -m paper_2606_13097_b200.build` (or __graft_entry__.build()); "
                                         "there is no CPU fallback")
        lib = C.CDLL(LIB_PATH)
        for name, (res, args) in SYMBOLS.items():
            fn = getattr(lib, name)
            fn.restype = res
            fn.argtypes = args
        _lib = lib
    return _lib


def _check(status: int):
    if status != FCG_OK:
        raise FcgError(status, load().fcg_last_error().decode())


def _ptr(x) -> int:
    if x is None:
        return None
    if isinstance(x, torch.Tensor):
        return x.data_ptr()
    if isinstance(x, np.ndarray):
        return x.ctypes.data
    return int(x)


def _stream(stream) -> int:
    if stream is None:
        return torch.cuda.current_stream().cuda_stream
    if isinstance(stream, torch.cuda.Stream):
        return stream.cuda_stream
    return int(stream)


def _i32(a) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(a, dtype=np.int32))


# ------------------------------------------------------------------------------------------------
# 1:1 functions
# ------------------------------------------------------------------------------------------------
def fcg_version() -> str:
    return load().fcg_version().decode()


def fcg_last_error() -> str:
    return load().fcg_last_error().decode()


def make_config(*, n_layers, n_q_heads, n_kv_heads, head_dim, page_size=16, rope_mode=FCG_ROPE_HALF_SPLIT,
                rope_base=1e4, inv_freq=None, arena=0, arena_bytes=0, max_segments=64, max_tasks=8,
                max_task_tokens=8192, n_pages=1024, workspace_bytes=0, device=0, host_arena=None, host_arena_bytes=0):
    cfg = fcg_config_t()
    cfg.host_arena, cfg.host_arena_bytes = _ptr(host_arena), int(host_arena_bytes)
    cfg.n_layers, cfg.n_q_heads, cfg.n_kv_heads, cfg.head_dim = n_layers, n_q_heads, n_kv_heads, head_dim
    cfg.page_size, cfg.rope_mode, cfg.rope_base = page_size, rope_mode, float(rope_base)
    keep = None
    if inv_freq is not None:
        keep = np.ascontiguousarray(np.asarray(inv_freq, dtype=np.float64))
        cfg.inv_freq = keep.ctypes.data_as(C.POINTER(C.c_double))
    cfg.arena, cfg.arena_bytes = _ptr(arena), int(arena_bytes)
    cfg.max_segments, cfg.max_tasks, cfg.max_task_tokens = max_segments, max_tasks, max_task_tokens
    cfg.n_pages, cfg.workspace_bytes, cfg.device = n_pages, workspace_bytes, device
    cfg._keepalive = keep
    return cfg


def fcg_arena_bytes_required(cfg: fcg_config_t, segment_tokens: int) -> int:
    return int(load().fcg_arena_bytes_required(C.byref(cfg), int(segment_tokens)))


def fcg_library_create(cfg: fcg_config_t) -> int:
    h = _P()
    _check(load().fcg_library_create(C.byref(cfg), C.byref(h)))
    return h.value


def fcg_library_destroy(handle: int) -> None:
    _check(load().fcg_library_destroy(handle))


def fcg_segment_register(handle, k, v, n_tokens, orig_start, strides=None, stream=None) -> int:
    sid = C.c_int32(-1)
    st = None
    if strides is not None:
        st = (C.c_int64 * 4)(*[int(s) for s in strides])
    _check(load().fcg_segment_register(handle, _ptr(k), _ptr(v), int(n_tokens), int(orig_start), st,
                                       _stream(stream), C.byref(sid)))
    return sid.value


def fcg_segment_register_fp8(handle, k, v, n_tokens, orig_start, strides=None, stream=None) -> int:
    sid = C.c_int32(-1)
    st = None
    if strides is not None:
        st = (C.c_int64 * 4)(*[int(s) for s in strides])
    _check(load().fcg_segment_register_fp8(handle, _ptr(k), _ptr(v), int(n_tokens), int(orig_start), st,
                                           _stream(stream), C.byref(sid)))
    return sid.value


def fcg_segment_storage(handle, seg_id):
    """-> (format, bytes)"""
    fmt, nbytes = C.c_int32(), C.c_uint64()
    _check(load().fcg_segment_storage(handle, int(seg_id), C.byref(fmt), C.byref(nbytes)))
    return fmt.value, nbytes.value


def fcg_segment_read(handle, seg_id, k_out, v_out, k_exp_out=None, v_exp_out=None, stream=None) -> None:
    _check(load().fcg_segment_read(handle, int(seg_id), _ptr(k_out), _ptr(v_out), _ptr(k_exp_out), _ptr(v_exp_out), _stream(stream)))


def fcg_segment_release(handle, seg_id) -> None:
    _check(load().fcg_segment_release(handle, int(seg_id)))


def _marshal_plans(plans):
    """plans: iterable of dicts {task_id, entries=[(seg, src_begin, n, dst)], holes=[(begin, n)], capacity_tokens}."""
    arr = (fcg_plan_t * len(plans))()
    keep = []
    for i, p in enumerate(plans):
        ents = p.get("entries", [])
        holes = p.get("holes", [])
        e_arr = (fcg_plan_entry_t * max(1, len(ents)))(*[fcg_plan_entry_t(*map(int, e)) for e in ents])
        h_arr = (fcg_hole_t * max(1, len(holes)))(*[fcg_hole_t(*map(int, h)) for h in holes])
        keep += [e_arr, h_arr]
        arr[i].task_id = int(p["task_id"])
        arr[i].entries = C.cast(e_arr, C.POINTER(fcg_plan_entry_t))
        arr[i].n_entries = len(ents)
        arr[i].holes = C.cast(h_arr, C.POINTER(fcg_hole_t))
        arr[i].n_holes = len(holes)
        arr[i].capacity_tokens = int(p.get("capacity_tokens", 0))
    return arr, keep


def fcg_stitch(handle, plans, stream=None) -> None:
    arr, _keep = _marshal_plans(list(plans))
    _check(load().fcg_stitch(handle, arr, len(arr), _stream(stream)))


def fcg_stitch_prefetch(handle, plans, stream=None) -> None:
    arr, _keep = _marshal_plans(list(plans))
    _check(load().fcg_stitch_prefetch(handle, arr, len(arr), _stream(stream)))


def fcg_patch(handle, task_id, layer_begin, n_layers, q, k, v, positions, out, stream=None) -> None:
    pos = _i32(positions)
    _check(load().fcg_patch(handle, int(task_id), int(layer_begin), int(n_layers), _ptr(q), _ptr(k), _ptr(v),
                            pos.ctypes.data_as(_PI), int(pos.size), _ptr(out), _stream(stream)))


def fcg_patch_rope(handle, task_id, layer_begin, n_layers, q, k, v, positions, out, stream=None) -> None:
    pos = np.ascontiguousarray(positions, dtype=np.int32)
    _check(load().fcg_patch_rope(handle, int(task_id), int(layer_begin), int(n_layers), _ptr(q), _ptr(k), _ptr(v),
                                 pos.ctypes.data_as(_PI), int(pos.size), _ptr(out), _stream(stream)))


def fcg_patch_host(handle, task_id, layer_begin, n_layers, q, k, v, positions, out, stream=None) -> None:
    pos = _i32(positions)
    _check(load().fcg_patch_host(handle, int(task_id), int(layer_begin), int(n_layers), _ptr(q), _ptr(k), _ptr(v),
                                 pos.ctypes.data_as(_PI), int(pos.size), _ptr(out), _stream(stream)))


def fcg_patch_batch(handle, task_ids, n_per_task, layer_begin, n_layers, q, k, v, positions, out, stream=None) -> None:
    ids, npt, pos = _i32(task_ids), _i32(n_per_task), _i32(positions)
    _check(load().fcg_patch_batch(handle, ids.ctypes.data_as(_PI), npt.ctypes.data_as(_PI), int(ids.size),
                                  int(layer_begin), int(n_layers), _ptr(q), _ptr(k), _ptr(v),
                                  pos.ctypes.data_as(_PI), _ptr(out), _stream(stream)))


def fcg_patch_batch_host(handle, task_ids, n_per_task, layer_begin, n_layers, q, k, v, positions, out, stream=None) -> None:
    ids, npt, pos = _i32(task_ids), _i32(n_per_task), _i32(positions)
    _check(load().fcg_patch_batch_host(handle, ids.ctypes.data_as(_PI), npt.ctypes.data_as(_PI), int(ids.size),
                                       int(layer_begin), int(n_layers), _ptr(q), _ptr(k), _ptr(v),
                                       pos.ctypes.data_as(_PI), _ptr(out), _stream(stream)))


def fcg_patch_plan_create(handle, task_ids, n_per_task, positions, layers_per_call, stream=None) -> int:
    ids, npt, pos = _i32(task_ids), _i32(n_per_task), _i32(positions)
    h = _P()
    _check(load().fcg_patch_plan_create(handle, ids.ctypes.data_as(_PI), npt.ctypes.data_as(_PI), int(ids.size),
                                        pos.ctypes.data_as(_PI), int(layers_per_call), _stream(stream), C.byref(h)))
    return h.value


def fcg_patch_planned(handle, plan, layer_begin, n_layers, q, k, v, out, stream=None) -> None:
    _check(load().fcg_patch_planned(handle, plan, int(layer_begin), int(n_layers), _ptr(q), _ptr(k), _ptr(v), _ptr(out),
                                    _stream(stream)))


def fcg_patch_plan_destroy(handle, plan) -> None:
    _check(load().fcg_patch_plan_destroy(handle, plan))


def fcg_task_page_table(handle, task_id):
    """-> (device pointer of int32 table, n_pages, n_tokens)"""
    p, n_pages, n_tokens = _P(), C.c_int32(), C.c_int32()
    _check(load().fcg_task_page_table(handle, int(task_id), C.byref(p), C.byref(n_pages), C.byref(n_tokens)))
    return p.value, n_pages.value, n_tokens.value


def fcg_task_page_table_host(handle, task_id) -> np.ndarray:
    n = C.c_int32()
    _check(load().fcg_task_page_table_host(handle, int(task_id), None, 0, C.byref(n)))
    out = np.empty(n.value, np.int32)
    _check(load().fcg_task_page_table_host(handle, int(task_id), out.ctypes.data_as(_PI), n.value, C.byref(n)))
    return out


def fcg_task_boundary_positions(handle, task_id, width) -> np.ndarray:
    n = C.c_int32()
    _check(load().fcg_task_boundary_positions(handle, int(task_id), int(width), None, 0, C.byref(n)))
    out = np.empty(n.value, np.int32)
    _check(load().fcg_task_boundary_positions(handle, int(task_id), int(width), out.ctypes.data_as(_PI), n.value, C.byref(n)))
    return out


def fcg_task_release(handle, task_id) -> None:
    _check(load().fcg_task_release(handle, int(task_id)))


def fcg_segment_offload(handle, seg_id, stream=None) -> None:
    _check(load().fcg_segment_offload(handle, int(seg_id), _stream(stream)))


def fcg_segment_prefetch(handle, seg_id, stream=None) -> None:
    _check(load().fcg_segment_prefetch(handle, int(seg_id), _stream(stream)))


def fcg_segment_info(handle, seg_id):
    n, o, r = C.c_int32(), C.c_int32(), C.c_int32()
    _check(load().fcg_segment_info(handle, int(seg_id), C.byref(n), C.byref(o), C.byref(r)))
    return n.value, o.value, bool(r.value)


def fcg_task_shift(handle, task_id, src_begin, n_tokens, dst_begin, stream=None) -> None:
    _check(load().fcg_task_shift(handle, int(task_id), int(src_begin), int(n_tokens), int(dst_begin), _stream(stream)))


def fcg_segment_extract(handle, task_id, begin, n_tokens, new_orig_start, stream=None) -> int:
    sid = C.c_int32(-1)
    _check(load().fcg_segment_extract(handle, int(task_id), int(begin), int(n_tokens), int(new_orig_start),
                                      _stream(stream), C.byref(sid)))
    return sid.value


def fcg_task_read(handle, task_id, layer, begin, n, k_out, v_out, stream=None) -> None:
    _check(load().fcg_task_read(handle, int(task_id), int(layer), int(begin), int(n), _ptr(k_out), _ptr(v_out),
                                _stream(stream)))


def fcg_segment_shift_static_max_tokens() -> int:
    return int(load().fcg_segment_shift_static_max_tokens())


def fcg_segment_shift_static(k_src, v_src, k_dst, v_dst, n_layers, n_kv_heads, n_tokens, head_dim, delta,
                             rope_mode=FCG_ROPE_HALF_SPLIT, rope_base=1e4, inv_freq=None, stream=None) -> None:
    """Re-rotate one dense segment [n_layers][n_kv_heads][n_tokens][head_dim] by `delta` positions (values copied)
    without allocating anything: for callers inside an engine that owns all device memory, or running while a graph
    capture forbids cudaMalloc.  The kernel's plan lives in a fixed array inside libfcg.so, one per GPU, so at most
    fcg_segment_shift_static_max_tokens() tokens per call and never two calls that can overlap on the device (keep them
    on one stream).  Buffers are on the CURRENT device.  Make the first call per device outside stream capture."""
    freq = None
    if inv_freq is not None:
        freq = np.ascontiguousarray(np.asarray(inv_freq, dtype=np.float64))
        assert freq.size == head_dim // 2
    _check(load().fcg_segment_shift_static(_ptr(k_src), _ptr(v_src), _ptr(k_dst), _ptr(v_dst), n_layers, n_kv_heads,
                                           n_tokens, head_dim, rope_mode, float(rope_base),
                                           None if freq is None else freq.ctypes.data_as(C.POINTER(C.c_double)),
                                           int(delta), _stream(stream)))


def fcg_pool_info(handle) -> dict:
    info = fcg_pool_info_t()
    _check(load().fcg_pool_info(handle, C.byref(info)))
    return {f: getattr(info, f) for f, _ in fcg_pool_info_t._fields_}


def fcg_set_attn_policy(handle, tc_min_rows: int, force_splits: int = 0) -> None:
    _check(load().fcg_set_attn_policy(handle, int(tc_min_rows), int(force_splits)))


def fcg_set_attn_pairs(handle, enable: bool) -> None:
    _check(load().fcg_set_attn_pairs(handle, 1 if enable else 0))


def fcg_set_attn_mixed(handle, enable: bool) -> None:
    _check(load().fcg_set_attn_mixed(handle, 1 if enable else 0))


def fcg_stats(handle) -> dict:
    st = fcg_stats_t()
    _check(load().fcg_stats(handle, C.byref(st)))
    return {f: getattr(st, f) for f, _ in fcg_stats_t._fields_}


class FcgScorer:
    """Locality score bookkeeping (Eq. 3, 8-10): host only, works without a GPU."""

    def __init__(self):
        h = _P()
        _check(load().fcg_scorer_create(C.byref(h)))
        self.handle = h.value

    def close(self):
        if getattr(self, "handle", None):
            load().fcg_scorer_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def record(self, trace) -> None:
        ids = np.ascontiguousarray(trace, dtype=np.int32)
        _check(load().fcg_scorer_record(self.handle, ids.ctypes.data_as(_PI), int(ids.size)))

    def set_ppl(self, fid, ppl) -> None:
        _check(load().fcg_scorer_set_ppl(self.handle, int(fid), float(ppl)))

    def forget(self, fid) -> None:
        _check(load().fcg_scorer_forget(self.handle, int(fid)))

    def score(self, fid, alpha, beta, gamma) -> float:
        out = C.c_double()
        _check(load().fcg_scorer_score(self.handle, int(fid), float(alpha), float(beta), float(gamma), C.byref(out)))
        return out.value

    def rank(self, ids, alpha, beta, gamma):
        ids = np.ascontiguousarray(ids, dtype=np.int32)
        out = np.empty_like(ids)
        sc = np.empty(ids.size, np.float64)
        _check(load().fcg_scorer_rank(self.handle, ids.ctypes.data_as(_PI), int(ids.size), float(alpha), float(beta),
                                      float(gamma), out.ctypes.data_as(_PI), sc.ctypes.data_as(C.POINTER(C.c_double))))
        return out.tolist(), sc.tolist()


# ------------------------------------------------------------------------------------------------
# convenience wrapper
# ------------------------------------------------------------------------------------------------
class FcgLibrary:
    """Owns a torch uint8 arena on ``device`` and a library handle over it."""

    def __init__(self, *, n_layers, n_q_heads, n_kv_heads, head_dim, page_size=16, rope_mode=FCG_ROPE_HALF_SPLIT,
                 rope_base=1e4, inv_freq=None, max_segments=64, max_tasks=8, max_task_tokens=8192, n_pages=1024,
                 workspace_bytes=0, segment_tokens=0, device=0, host_tier_tokens=0):
        self.n_layers, self.n_q_heads, self.n_kv_heads, self.head_dim = n_layers, n_q_heads, n_kv_heads, head_dim
        self.page_size = page_size
        self.device = torch.device("cuda", device)
        # second tier (Eq. 3): a pinned host tensor for `host_tier_tokens` tokens of offloaded segments
        self.host_arena = None
        if host_tier_tokens > 0:
            nbytes = host_tier_tokens * n_layers * n_kv_heads * head_dim * 4 + 512 * (max_segments + 1)
            self.host_arena = torch.empty(nbytes + 256, dtype=torch.uint8).pin_memory()
        hptr = 0 if self.host_arena is None else (self.host_arena.data_ptr() + 255) // 256 * 256
        cfg = make_config(n_layers=n_layers, n_q_heads=n_q_heads, n_kv_heads=n_kv_heads, head_dim=head_dim,
                          page_size=page_size, rope_mode=rope_mode, rope_base=rope_base, inv_freq=inv_freq,
                          max_segments=max_segments, max_tasks=max_tasks, max_task_tokens=max_task_tokens,
                          n_pages=n_pages, workspace_bytes=workspace_bytes, device=device,
                          host_arena=hptr or None,
                          host_arena_bytes=0 if self.host_arena is None else self.host_arena.numel() - 256)
        need = fcg_arena_bytes_required(cfg, segment_tokens)
        if need == 0:
            raise FcgError(FCG_ERR_INVALID_ARG, "bad configuration")
        self.arena = torch.empty(need, dtype=torch.uint8, device=self.device)
        cfg.arena, cfg.arena_bytes = self.arena.data_ptr(), need
        self.handle = fcg_library_create(cfg)

    def close(self):
        if getattr(self, "handle", None):
            fcg_library_destroy(self.handle)
            self.handle = None
            self.arena = None
            self.host_arena = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def segment_register(self, k: torch.Tensor, v: torch.Tensor, orig_start: int, stream=None) -> int:
        assert k.dtype == torch.bfloat16 and v.dtype == torch.bfloat16 and k.is_cuda and v.is_cuda
        assert k.shape == v.shape and k.stride() == v.stride()
        return fcg_segment_register(self.handle, k, v, k.shape[2], orig_start, k.stride(), stream)

    def segment_register_fp8(self, k: torch.Tensor, v: torch.Tensor, orig_start: int, stream=None) -> int:
        assert k.dtype == torch.bfloat16 and v.dtype == torch.bfloat16 and k.is_cuda and v.is_cuda
        assert k.shape == v.shape and k.stride() == v.stride()
        return fcg_segment_register_fp8(self.handle, k, v, k.shape[2], orig_start, k.stride(), stream)

    def segment_storage(self, seg_id):
        return fcg_segment_storage(self.handle, seg_id)

    def segment_read(self, seg_id, stream=None):
        """the stored representation: (k, v) bf16 tensors, or (k codes, v codes, k scale bytes, v scale bytes) uint8"""
        n, _, _ = fcg_segment_info(self.handle, seg_id)
        fmt, _ = fcg_segment_storage(self.handle, seg_id)
        shape = (self.n_layers, self.n_kv_heads, n, self.head_dim)
        if fmt == FCG_STORE_FP8_E4M3:
            k, v = torch.empty(shape, dtype=torch.uint8, device=self.device), torch.empty(shape, dtype=torch.uint8, device=self.device)
            ke, ve = torch.empty(shape[:3], dtype=torch.uint8, device=self.device), torch.empty(shape[:3], dtype=torch.uint8, device=self.device)
            fcg_segment_read(self.handle, seg_id, k, v, ke, ve, stream)
            return k, v, ke, ve
        k, v = torch.empty(shape, dtype=torch.bfloat16, device=self.device), torch.empty(shape, dtype=torch.bfloat16, device=self.device)
        fcg_segment_read(self.handle, seg_id, k, v, None, None, stream)
        return k, v

    def segment_release(self, seg_id):
        fcg_segment_release(self.handle, seg_id)

    def segment_offload(self, seg_id, stream=None):
        fcg_segment_offload(self.handle, seg_id, stream)

    def segment_prefetch(self, seg_id, stream=None):
        fcg_segment_prefetch(self.handle, seg_id, stream)

    def segment_info(self, seg_id):
        return fcg_segment_info(self.handle, seg_id)

    def stitch(self, plans, stream=None):
        fcg_stitch(self.handle, plans, stream)

    def stitch_prefetch(self, plans, stream=None):
        fcg_stitch_prefetch(self.handle, plans, stream)

    def patch(self, task_id, layer_begin, q, k, v, positions, out=None, stream=None) -> torch.Tensor:
        assert q.is_cuda and q.is_contiguous() and k.is_contiguous() and v.is_contiguous()
        if out is None:
            out = torch.empty_like(q)
        fcg_patch(self.handle, task_id, layer_begin, q.shape[0], q, k, v, positions, out, stream)
        return out

    def patch_rope(self, task_id, layer_begin, q, k, v, positions, out=None, stream=None) -> torch.Tensor:
        assert q.is_cuda and q.is_contiguous() and k.is_contiguous() and v.is_contiguous()
        if out is None:
            out = torch.empty_like(q)
        fcg_patch_rope(self.handle, task_id, layer_begin, q.shape[0], q, k, v, positions, out, stream)
        return out

    def patch_host(self, task_id, layer_begin, q, k, v, positions, out, stream=None) -> torch.Tensor:
        assert not q.is_cuda and q.is_contiguous() and k.is_contiguous() and v.is_contiguous() and out.is_contiguous()
        fcg_patch_host(self.handle, task_id, layer_begin, q.shape[0], q, k, v, positions, out, stream)
        return out

    def patch_batch(self, task_ids, n_per_task, layer_begin, q, k, v, positions, out=None, stream=None) -> torch.Tensor:
        if out is None:
            out = torch.empty_like(q)
        fcg_patch_batch(self.handle, task_ids, n_per_task, layer_begin, q.shape[0], q, k, v, positions, out, stream)
        return out

    def patch_batch_host(self, task_ids, n_per_task, layer_begin, q, k, v, positions, out, stream=None) -> torch.Tensor:
        assert not q.is_cuda and q.is_contiguous() and k.is_contiguous() and v.is_contiguous() and out.is_contiguous()
        fcg_patch_batch_host(self.handle, task_ids, n_per_task, layer_begin, q.shape[0], q, k, v, positions, out, stream)
        return out

    def patch_plan_create(self, task_ids, n_per_task, positions, layers_per_call, stream=None) -> int:
        return fcg_patch_plan_create(self.handle, task_ids, n_per_task, positions, layers_per_call, stream)

    def patch_planned(self, plan, layer_begin, q, k, v, out, stream=None) -> torch.Tensor:
        fcg_patch_planned(self.handle, plan, layer_begin, q.shape[0], q, k, v, out, stream)
        return out

    def patch_plan_destroy(self, plan) -> None:
        fcg_patch_plan_destroy(self.handle, plan)

    def task_page_table(self, task_id):
        return fcg_task_page_table(self.handle, task_id)

    def task_page_table_host(self, task_id) -> np.ndarray:
        return fcg_task_page_table_host(self.handle, task_id)

    def task_read(self, task_id, layer, begin, n, stream=None):
        k = torch.empty((self.n_kv_heads, n, self.head_dim), dtype=torch.bfloat16, device=self.device)
        v = torch.empty_like(k)
        fcg_task_read(self.handle, task_id, layer, begin, n, k, v, stream)
        return k, v

    def task_release(self, task_id):
        fcg_task_release(self.handle, task_id)

    def task_boundary_positions(self, task_id, width) -> np.ndarray:
        return fcg_task_boundary_positions(self.handle, task_id, width)

    def task_shift(self, task_id, src_begin, n_tokens, dst_begin, stream=None):
        fcg_task_shift(self.handle, task_id, src_begin, n_tokens, dst_begin, stream)

    def segment_extract(self, task_id, begin, n_tokens, new_orig_start, stream=None) -> int:
        return fcg_segment_extract(self.handle, task_id, begin, n_tokens, new_orig_start, stream)

    def pool_info(self) -> dict:
        return fcg_pool_info(self.handle)

    def stats(self) -> dict:
        return fcg_stats(self.handle)

    def set_attn_policy(self, tc_min_rows: int, force_splits: int = 0) -> None:
        fcg_set_attn_policy(self.handle, tc_min_rows, force_splits)

    def set_attn_pairs(self, enable: bool) -> None:
        fcg_set_attn_pairs(self.handle, enable)

    def set_attn_mixed(self, enable: bool) -> None:
        fcg_set_attn_mixed(self.handle, enable)
