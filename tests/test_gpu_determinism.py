"""Race detection by repetition ("race detection / sanitizers"; compute-sanitizer is closed on this pool,
profiles/r02_sanitizer.md): every kernel of the graft path is free of atomics and of data-dependent scheduling, so the same
call on the same inputs must give the same BITS every time.  A missing barrier or fence in the mbarrier / TMEM pipelines
(the stage rings, the S / P hand-over, the O rescale, the stream merge, the split-KV combine) shows up as a run that differs.
Each case runs one stitch + patch once against the oracle and then repeats the patch, with hundreds of CTAs in flight so that
CTAs of different progress share SMs, and compares the outputs and the scattered cache rows bit for bit."""
import numpy as np
import pytest
import torch

from paper_2606_13097_b200 import synth
import fcg_testlib as T

pytestmark = pytest.mark.gpu

REPEATS = 25

CASES = [
    # n, Hq, Hkv, D, ctx, forced splits: the CTA classes of both head dims, with and without the combine kernel
    (1, 8, 8, 128, 3000, 0), (1, 8, 2, 128, 3000, 5), (16, 8, 8, 128, 2100, 0), (48, 8, 4, 128, 1777, 3),
    (100, 4, 4, 128, 1500, 0), (33, 16, 4, 128, 1900, 2), (300, 4, 2, 128, 1400, 0), (200, 8, 4, 128, 900, 3),
    (1, 8, 8, 64, 3000, 0), (20, 8, 4, 64, 2500, 4), (120, 4, 4, 64, 1500, 0), (260, 4, 2, 64, 1000, 2),
    (1, 4, 2, 256, 3000, 0), (20, 8, 4, 256, 2500, 3), (128, 2, 2, 256, 1500, 0), (300, 4, 2, 256, 700, 2),
]


@pytest.mark.parametrize("n,Hq,Hkv,D,ctx,splits", CASES)
def test_repeated_patch_calls_are_bit_identical(n, Hq, Hkv, D, ctx, splits):
    L, P = 6, 16
    cfg = synth.GraftConfig("det", L, Hq, Hkv, D, P, 1e4, 3, ctx // 3 + 1, ctx // 3 + 60, 4000, 1, 3, 3, 0, holes=((-1, n),))
    wl = synth.make_workload(cfg, n + ctx + D)
    orc, lib, seg_ids = T.make_pair(cfg, wl, 4, workspace_bytes=256 << 20)
    c_plans, o_plans = T.plans_of(wl, seg_ids)
    orc.stitch(o_plans)
    lib.stitch(c_plans)
    lib.set_attn_policy(1, splits)
    task = wl.tasks[0]
    out, ref = T.run_patch_both(orc, lib, cfg, task, 9)
    T.assert_attn_close(out, ref, "first run")
    first = synth.to_bits(out).copy()
    q, k, v = [x.cuda().contiguous() for x in synth.patch_qkv(cfg, task.task_id, len(task.positions), 9, "cpu")]
    cache0 = [tuple(synth.to_bits(x).copy() for x in lib.task_read(0, layer, 0, task.capacity)) for layer in (0, L - 1)]
    outs = [lib.patch(0, 0, q, k, v, task.positions) for _ in range(REPEATS)]
    torch.cuda.synchronize()
    for i, o in enumerate(outs):
        assert np.array_equal(synth.to_bits(o), first), f"run {i + 2} of the same patch differs from the first"
    for (kb, vb), layer in zip(cache0, (0, L - 1)):
        k2, v2 = lib.task_read(0, layer, 0, task.capacity)
        assert np.array_equal(synth.to_bits(k2), kb) and np.array_equal(synth.to_bits(v2), vb), "cache rows changed between runs"
    lib.close()


@pytest.mark.parametrize("D", [64, 128, 256])
def test_repeated_stitch_calls_are_bit_identical(D):
    """the gather kernel, bf16 and fp8 sources, writes the same bits on every run (release + stitch again reuses the pages
    in the same order: LIFO pool, R9)"""
    cfg = synth.GraftConfig("detst", 4, 4, 2, D, 16, 5e5, 8, 100, 400, 5000, 2, 4, 5, 0, distinct_segments=False)
    wl = synth.make_workload(cfg, 21)
    orc, lib, seg_ids = T.make_pair(cfg, wl, 21)
    c_plans, o_plans = T.plans_of(wl, seg_ids)
    orc.stitch(o_plans)
    lib.stitch(c_plans)
    T.compare_stitched(orc, lib, wl)
    snap = {t.task_id: [tuple(synth.to_bits(x).copy() for x in lib.task_read(t.task_id, layer, 0, t.capacity)) for layer in range(cfg.n_layers)]
            for t in wl.tasks}
    tables = {t.task_id: lib.task_page_table_host(t.task_id).copy() for t in wl.tasks}
    for _ in range(8):
        for t in reversed(wl.tasks):
            lib.task_release(t.task_id)
        lib.stitch(c_plans)
        torch.cuda.synchronize()
        for t in wl.tasks:
            assert np.array_equal(lib.task_page_table_host(t.task_id), tables[t.task_id])
            filled = orc.tasks[t.task_id].filled
            for layer in range(cfg.n_layers):
                k2, v2 = lib.task_read(t.task_id, layer, 0, t.capacity)
                assert np.array_equal(synth.to_bits(k2)[:, filled], snap[t.task_id][layer][0][:, filled])
                assert np.array_equal(synth.to_bits(v2)[:, filled], snap[t.task_id][layer][1][:, filled])
    lib.close()
