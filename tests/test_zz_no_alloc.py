"""fcg_segment_shift_static: the key re-rotation of cache-stitching for callers that cannot allocate device memory --
a plug-in inside a serving engine that took all of HBM for its own pool, or code running while another thread's graph
capture makes the CUDA runtime refuse cudaMalloc.  Its kernel plan lives in a fixed array inside libfcg.so (one per
GPU, 65 536 tokens per call at most) instead of in an arena workspace.

The check is against the library's ordinary path, bit for bit: register the same segment, fcg_stitch it `delta`
positions away from where it was encoded, read the task's cache back.  Two calls are issued back to back on one stream
with nothing in between (the second is shorter and has another delta, so whatever the first left in the shared array
beyond the second's plan must not matter), then a third with a run-time head_dim and interleaved pairs.

This file is named to be collected last: `pytest -x` stops at the first failure, and a failure here must not hide the
parity tests.  It passes alone in a fresh process (the first call then does the per-device set-up) and after the rest.
"""
import numpy as np
import pytest
import torch

from paper_2606_13097_b200 import binding as B


def _segment(n_layers, n_kv_heads, n, head_dim, seed):
    g = torch.Generator().manual_seed(seed)
    k = torch.randn(n_layers, n_kv_heads, n, head_dim, generator=g).to(torch.bfloat16).cuda()
    v = torch.randn(n_layers, n_kv_heads, n, head_dim, generator=g).to(torch.bfloat16).cuda()
    return k, v


def _stitched_by_library(lib, k, v, orig_start, delta, task_id):
    """the existing path: segment -> fcg_stitch at orig_start + delta -> dense read-back [L][Hkv][n][D]"""
    n = k.shape[2]
    dst = orig_start + delta
    seg = lib.segment_register(k, v, orig_start)
    lib.stitch([{"task_id": task_id, "entries": [(seg, 0, n, dst)], "holes": [(0, dst)] if dst else [],
                 "capacity_tokens": dst + n}])
    ks, vs = zip(*[lib.task_read(task_id, layer, dst, n) for layer in range(lib.n_layers)])
    return torch.stack(ks), torch.stack(vs)


def _same_bits(a, b):
    return torch.equal(a.contiguous().view(torch.int16), b.contiguous().view(torch.int16))


@pytest.mark.gpu
def test_two_calls_in_a_row_match_the_library_path():
    L, Hq, Hkv, D, base = 3, 4, 2, 128, 5e5
    n1, d1, n2, d2 = 1237, 4321, 301, -257          # ragged lengths: 78 and 19 chunks, the last ones partial
    k1, v1 = _segment(L, Hkv, n1, D, 11)
    k2, v2 = _segment(L, Hkv, n2, D, 12)
    lib = B.FcgLibrary(n_layers=L, n_q_heads=Hq, n_kv_heads=Hkv, head_dim=D, rope_base=base, max_segments=4, max_tasks=2,
                       max_task_tokens=8192, n_pages=512, segment_tokens=n1 + n2)
    want_k1, want_v1 = _stitched_by_library(lib, k1, v1, 0, d1, 0)
    want_k2, want_v2 = _stitched_by_library(lib, k2, v2, 300, d2, 1)

    got = [torch.full_like(t, float("nan")) for t in (k1, v1, k2, v2)]
    torch.cuda.synchronize()
    B.fcg_segment_shift_static(k1, v1, got[0], got[1], L, Hkv, n1, D, d1, rope_base=base)
    free_before = torch.cuda.mem_get_info()[0]
    B.fcg_segment_shift_static(k2, v2, got[2], got[3], L, Hkv, n2, D, d2, rope_base=base)   # no sync in between
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before, "the call changed the amount of free device memory"
    assert _same_bits(got[0], want_k1) and _same_bits(got[1], want_v1), "first call differs from fcg_stitch"
    assert _same_bits(got[2], want_k2) and _same_bits(got[3], want_v2), "second call differs from fcg_stitch"
    assert _same_bits(got[1], v1) and _same_bits(got[3], v2)            # values are bit copies
    assert not _same_bits(got[0], k1)                                   # and the keys really were rotated

    # delta 0: keys are copied too; and the first call's result is reproduced after the array held other plans
    out_k, out_v = torch.empty_like(k2), torch.empty_like(v2)
    B.fcg_segment_shift_static(k2, v2, out_k, out_v, L, Hkv, n2, D, 0, rope_base=base)
    again_k, again_v = torch.empty_like(k1), torch.empty_like(v1)
    B.fcg_segment_shift_static(k1, v1, again_k, again_v, L, Hkv, n1, D, d1, rope_base=base)
    torch.cuda.synchronize()
    assert _same_bits(out_k, k2) and _same_bits(out_v, v2)
    assert _same_bits(again_k, want_k1) and _same_bits(again_v, want_v1)
    lib.close()


@pytest.mark.gpu
def test_runtime_head_dim_interleaved_and_given_frequencies():
    L, Hq, Hkv, D, n, delta = 2, 6, 3, 80, 530, 77
    inv_freq = 1.0 / (1e4 ** (np.arange(D // 2, dtype=np.float64) * 2 / D)) * 0.5      # a scaled-RoPE style table
    k, v = _segment(L, Hkv, n, D, 13)
    lib = B.FcgLibrary(n_layers=L, n_q_heads=Hq, n_kv_heads=Hkv, head_dim=D, rope_mode=B.FCG_ROPE_INTERLEAVED,
                       inv_freq=inv_freq, max_segments=2, max_tasks=1, max_task_tokens=1024, n_pages=64, segment_tokens=n)
    want_k, want_v = _stitched_by_library(lib, k, v, 5, delta, 0)
    got_k, got_v = torch.empty_like(k), torch.empty_like(v)
    B.fcg_segment_shift_static(k, v, got_k, got_v, L, Hkv, n, D, delta, rope_mode=B.FCG_ROPE_INTERLEAVED, inv_freq=inv_freq)
    torch.cuda.synchronize()
    assert _same_bits(got_k, want_k) and _same_bits(got_v, want_v)
    lib.close()


def test_sizes_beyond_the_static_plan_are_refused():
    """host-side checks only (they come before any CUDA call, so this runs without a GPU)"""
    limit = B.fcg_segment_shift_static_max_tokens()
    assert limit == 65536
    with pytest.raises(B.FcgError) as e:
        B.fcg_segment_shift_static(256, 512, 768, 1024, 1, 1, limit + 1, 128, 5, stream=0)
    assert e.value.status == B.FCG_ERR_RANGE and str(limit) in str(e.value)
    with pytest.raises(B.FcgError) as e:                                   # k_dst == k_src
        B.fcg_segment_shift_static(4096, 1 << 20, 4096, 2 << 20, 1, 1, 16, 128, 5, stream=0)
    assert e.value.status == B.FCG_ERR_OVERLAP
    for bad in (dict(head_dim=72), dict(n_layers=0), dict(rope_base=0.0)):
        args = dict(n_layers=1, n_kv_heads=1, n_tokens=16, head_dim=128, delta=5, rope_base=1e4, stream=0)
        args.update(bad)
        with pytest.raises(B.FcgError) as e:
            B.fcg_segment_shift_static(4096, 1 << 20, 2 << 20, 3 << 20, **args)
        assert e.value.status == B.FCG_ERR_INVALID_ARG, bad
    B.fcg_segment_shift_static(0, 0, 0, 0, 1, 1, 0, 128, 5, stream=0)        # an empty segment is a no-op
