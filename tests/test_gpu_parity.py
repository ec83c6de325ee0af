"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the same
seeded inputs.  Bars (BASELINE.json north_star): page tables, V gather, scatter bit-exact; shifted K
within 1 bf16 ulp of the fp64-computed, bf16-rounded reference for EVERY element; patch attention
within 2e-2 relative + 1e-2 absolute."""
import numpy as np
import pytest
import torch

from oracle import fcg_oracle as O
from paper_2606_13097_b200 import synth
import fcg_testlib as T

pytestmark = pytest.mark.gpu


def _binding():
    from paper_2606_13097_b200 import binding
    return binding


# ------------------------------------------------------------------------------------------------
# C1 (BASELINE.json configs[0]) end to end, seeds 1, 2, 3 (the paper's seeds)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("seed", [1, 2, 3])
def test_c1_stitch_and_patch(seed):
    cfg = synth.C1
    wl = synth.make_workload(cfg, seed)
    orc, lib, seg_ids = T.make_pair(cfg, wl, seed, only_segments=list(range(cfg.n_segments)))
    c_plans, o_plans = T.plans_of(wl, seg_ids)
    orc.stitch(o_plans)
    lib.stitch(c_plans)
    hist = T.compare_stitched(orc, lib, wl)
    assert hist[0] > 0.99 * hist.sum()
    task = wl.tasks[0]
    out, ref = T.run_patch_both(orc, lib, cfg, task, seed)
    T.assert_attn_close(out, ref, "C1 mid patch")
    T.compare_cache_bits(orc, lib, task.task_id, task.positions)
    assert lib.stats()["last_attn_path"] in (1, 2)
    # variant b: 32 more tokens can NOT be appended beyond capacity
    with pytest.raises(_binding().FcgError) as e:
        lib.patch(0, 0, *[x.cuda() for x in synth.patch_qkv(cfg, 0, 1, seed)], [task.capacity])
    assert e.value.status == _binding().FCG_ERR_RANGE
    lib.close()


def test_c1_appended_patch_and_retry_overwrite():
    """patch at the end of the cache (Eq. 4 case), then a second call over the same positions (retry)."""
    cfg = synth.scaled(synth.C1, holes=((1, 32), (-1, 32)))
    wl = synth.make_workload(cfg, 2)
    orc, lib, seg_ids = T.make_pair(cfg, wl, 2)
    c_plans, o_plans = T.plans_of(wl, seg_ids)
    orc.stitch(o_plans)
    lib.stitch(c_plans)
    task = wl.tasks[0]
    mid = np.arange(task.holes[0][0], task.holes[0][0] + 32, dtype=np.int32)
    end = np.arange(task.holes[1][0], task.holes[1][0] + 32, dtype=np.int32)
    bnd = _binding()
    with pytest.raises(bnd.FcgError) as e:          # end patch first would attend over the unfilled mid hole
        lib.patch(0, 0, *[x.cuda() for x in synth.patch_qkv(cfg, 0, 32, 9)], end)
    assert e.value.status == bnd.FCG_ERR_UNFILLED
    with pytest.raises(O.OracleError) as eo:
        orc.patch(0, 0, *[synth.to_bits(x) for x in synth.patch_qkv(cfg, 0, 32, 9)], end)
    assert eo.value.status == e.value.status
    out, ref = T.run_patch_both(orc, lib, cfg, task, 3, positions=mid)
    T.assert_attn_close(out, ref, "mid")
    out, ref = T.run_patch_both(orc, lib, cfg, task, 4, positions=end)
    T.assert_attn_close(out, ref, "end")
    out, ref = T.run_patch_both(orc, lib, cfg, task, 5, positions=np.concatenate([mid[5:9], end[-3:]]))
    T.assert_attn_close(out, ref, "retry")
    T.compare_cache_bits(orc, lib, 0, np.concatenate([mid, end]))
    lib.close()


# ------------------------------------------------------------------------------------------------
# geometry sweep: head_dim, page size, GQA group, ragged chunks, deltas of both signs, sub-ranges
# ------------------------------------------------------------------------------------------------
GEOMS = [
    # L, Hq, Hkv, D, P, base
    (2, 4, 4, 128, 16, 1e4),
    (2, 8, 2, 128, 16, 5e5),
    (1, 8, 1, 128, 64, 1e6),
    (3, 6, 3, 64, 8, 1e4),
    (1, 16, 2, 64, 32, 1e4),
    # head_dim 256 (Gemma-style heads, R27): one CTA class on the tcgen05 path, stitch_kernel<256>
    (2, 8, 2, 256, 16, 1e4),
    (1, 4, 4, 256, 64, 5e5),
    (1, 6, 3, 256, 8, 1e6),
    # other multiples of 16 (R27): run-time-D gather kernel, tcgen05 attention at the next instantiated width with zero padding
    (2, 4, 2, 96, 16, 1e4),
    (1, 8, 2, 80, 32, 5e5),
    (1, 4, 4, 192, 16, 1e4),
    (2, 6, 3, 160, 8, 1e4),
    (1, 2, 2, 32, 16, 1e4),
    (1, 4, 1, 112, 64, 1e4),
    (1, 2, 1, 224, 16, 1e6),
    (1, 4, 2, 16, 16, 1e4),
    (1, 2, 2, 48, 8, 1e4),
]


@pytest.mark.parametrize("geom", GEOMS)
def test_geometry_sweep(geom):
    L, Hq, Hkv, D, P, base = geom
    cfg = synth.GraftConfig("sweep", L, Hq, Hkv, D, P, base, 10, 5, 211, 5000, 1, 5, 5, 0,
                            holes=((0, 3), (2, 17), (-1, 9)))
    wl = synth.make_workload(cfg, 7)
    orc, lib, seg_ids = T.make_pair(cfg, wl, 7)
    c_plans, o_plans = T.plans_of(wl, seg_ids)
    orc.stitch(o_plans)
    lib.stitch(c_plans)
    T.compare_stitched(orc, lib, wl)
    task = wl.tasks[0]
    # three calls: each hole separately (later calls see earlier patches)
    for hi, (b, n) in enumerate(sorted(task.holes)):
        pos = np.arange(b, b + n, dtype=np.int32)
        out, ref = T.run_patch_both(orc, lib, cfg, task, 20 + hi, positions=pos)
        T.assert_attn_close(out, ref, f"hole {hi} geom {geom}")
    T.compare_cache_bits(orc, lib, 0, task.positions)
    lib.close()


def test_identity_graft_is_bit_exact_and_rope_none():
    """P2: one segment grafted at delta 0 equals the original (K and V); rope_mode NONE is a pure gather."""
    cfg = synth.GraftConfig("ident", 2, 4, 2, 128, 16, 1e4, 2, 100, 100, 0, 1, 1, 1, 0)
    wl = synth.make_workload(cfg, 1)
    wl.orig_starts[:] = [37, 0]
    wl.tasks[0].entries = [(0, 0, 100, 37)]
    wl.tasks[0].capacity = 137
    wl.tasks[0].holes = []
    orc, lib, seg_ids = T.make_pair(cfg, wl, 1)
    c_plans, o_plans = T.plans_of(wl, seg_ids)
    orc.stitch(o_plans)
    lib.stitch(c_plans)
    k0, v0 = synth.segment_kv(cfg, 0, 100, 1)
    for layer in range(2):
        k, v = lib.task_read(0, layer, 37, 100)
        assert torch.equal(k.cpu(), k0[layer]) and torch.equal(v.cpu(), v0[layer])
    lib.close()
    for mode in (0,):
        orc, lib, seg_ids = T.make_pair(cfg, wl, 1, rope_mode=mode)
        wl.tasks[0].entries = [(0, 10, 80, 3)]
        wl.tasks[0].capacity = 83
        c_plans, o_plans = T.plans_of(wl, seg_ids)
        orc.stitch(o_plans)
        lib.stitch(c_plans)
        k, v = lib.task_read(0, 1, 3, 80)
        assert torch.equal(k.cpu(), k0[1][:, 10:90]) and torch.equal(v.cpu(), v0[1][:, 10:90])
        lib.close()


def test_scaled_rope_inv_freq_override_and_large_deltas():
    """inv_freq override (scaled RoPE, DESIGN R3) and |delta| up to ~32k, both signs."""
    D = 128
    inv = O.rope_inv_freq(D, 5e5) / np.where(np.arange(D // 2) > 40, 8.0, 1.0)
    cfg = synth.GraftConfig("scaled", 1, 2, 2, D, 16, 5e5, 4, 300, 400, 32768, 1, 4, 4, 0)
    wl = synth.make_workload(cfg, 3)
    wl.orig_starts[:] = [0, 32768, 20000, 5]
    t = wl.tasks[0]
    t.entries = [(0, 0, 300, 31000), (1, 0, 300, 0), (2, 7, 250, 300), (3, 0, 300, 600)]
    t.holes, t.capacity, t.positions = [], 31300, np.zeros(0, np.int32)
    orc, lib, seg_ids = T.make_pair(cfg, wl, 3, inv_freq=inv, only_segments=[0, 1, 2, 3])
    c_plans, o_plans = T.plans_of(wl, seg_ids)
    orc.stitch(o_plans)
    lib.stitch(c_plans)
    assert orc.tasks[0].deltas == [31000, -32768, 300 - 20000 - 7, 595]
    T.compare_stitched(orc, lib, wl)
    lib.close()


# ------------------------------------------------------------------------------------------------
# attention special cases on the GPU
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n,Hq,Hkv,D", [(1, 4, 4, 128), (45, 6, 2, 128), (64, 8, 8, 64), (130, 2, 2, 128), (5, 32, 4, 128)])
def test_p12_empty_cache_patch_is_causal_self_attention(n, Hq, Hkv, D):
    """empty cache + one patch covering [0, n): oracle == causal self-attention (pinned vs torch SDPA on the
    CPU side); the GPU must match, for row counts that hit every row-block variant."""
    cfg = synth.GraftConfig("selfattn", 2, Hq, Hkv, D, 16, 1e4, 1, 8, 8, 0, 1, 0, 0, 0, holes=((-1, n),))
    wl = synth.make_workload(cfg, 1)
    wl.tasks[0].entries = []
    orc, lib, seg_ids = T.make_pair(cfg, wl, 1, only_segments=[])
    c_plans, o_plans = T.plans_of(wl, seg_ids)
    orc.stitch(o_plans)
    lib.stitch(c_plans)
    out, ref = T.run_patch_both(orc, lib, cfg, wl.tasks[0], 11)
    T.assert_attn_close(out, ref, f"self-attention n={n}")
    lib.close()


def test_long_cache_forces_kv_splits_and_matches():
    """few heads, one layer, long cache -> the split-KV + combine path; also non-multiple-of-tile lengths."""
    cfg = synth.GraftConfig("long", 1, 4, 1, 128, 16, 1e4, 6, 900, 1100, 4000, 1, 6, 6, 0,
                            holes=((2, 5), (-1, 11)))
    wl = synth.make_workload(cfg, 5)
    orc, lib, seg_ids = T.make_pair(cfg, wl, 5)
    c_plans, o_plans = T.plans_of(wl, seg_ids)
    orc.stitch(o_plans)
    lib.stitch(c_plans)
    T.compare_stitched(orc, lib, wl)
    out, ref = T.run_patch_both(orc, lib, cfg, wl.tasks[0], 6)
    assert lib.stats()["last_attn_splits"] > 1
    T.assert_attn_close(out, ref, "split-KV")
    lib.close()


def test_p10_causality_on_gpu():
    """changing K/V at positions > p_i leaves output i bit-identical (same launch shape)."""
    cfg = synth.GraftConfig("causal", 1, 4, 2, 128, 16, 1e4, 3, 200, 300, 100, 1, 3, 3, 0, holes=((0, 8), (-1, 8)))
    outs = []
    for variant in range(2):
        wl = synth.make_workload(cfg, 4)
        orc, lib, seg_ids = T.make_pair(cfg, wl, 4)
        c_plans, _ = T.plans_of(wl, seg_ids)
        lib.stitch(c_plans)
        task = wl.tasks[0]
        q, k, v = [x.cuda() for x in synth.patch_qkv(cfg, 0, 16, 4)]
        if variant:   # perturb only the END patch's k/v: rows of the mid patch must not notice
            k[:, 8:] = k[:, 8:] * 2
            v[:, 8:] = v[:, 8:] + 1
        outs.append(lib.patch(0, 0, q, k, v, task.positions).cpu())
        lib.close()
    assert torch.equal(outs[0][:, :8], outs[1][:, :8])
    assert not torch.equal(outs[0][:, 8:], outs[1][:, 8:])


def test_patch_host_and_batch_variants_match_device_call():
    cfg = synth.GraftConfig("variants", 2, 8, 2, 128, 16, 1e4, 12, 64, 300, 3000, 3, 2, 4, 0,
                            total_min=200, total_max=1200, distinct_segments=False,
                            holes=((-1, 0),), patch_min=3, patch_max=40)
    wl = synth.make_workload(cfg, 8)
    orc, lib, seg_ids = T.make_pair(cfg, wl, 8, only_segments=list(range(12)))
    c_plans, o_plans = T.plans_of(wl, seg_ids)
    orc.stitch(o_plans)
    lib.stitch(c_plans)              # one call, 3 plans
    T.compare_stitched(orc, lib, wl)
    # batched patch of all three tasks
    qs, ks, vs, refs = [], [], [], []
    for t in wl.tasks:
        q, k, v = synth.patch_qkv(cfg, t.task_id, len(t.positions), 8)
        refs.append(orc.patch(t.task_id, 0, synth.to_bits(q), synth.to_bits(k), synth.to_bits(v), t.positions))
        qs.append(q), ks.append(k), vs.append(v)
    q = torch.cat(qs, dim=1).cuda().contiguous()
    k = torch.cat(ks, dim=1).cuda().contiguous()
    v = torch.cat(vs, dim=1).cuda().contiguous()
    out = lib.patch_batch([t.task_id for t in wl.tasks], [len(t.positions) for t in wl.tasks], 0, q, k, v,
                          np.concatenate([t.positions for t in wl.tasks]))
    torch.cuda.synchronize()
    T.assert_attn_close(out, np.concatenate(refs, axis=1), "batched patch")
    for t in wl.tasks:
        T.compare_cache_bits(orc, lib, t.task_id, t.positions)
    # host-buffer call == device call (re-patching task 0 with the same tensors)
    t0 = wl.tasks[0]
    qh, kh, vh = [x.contiguous().pin_memory() for x in (qs[0], ks[0], vs[0])]
    oh = torch.empty_like(qh).pin_memory()
    lib.patch_host(0, 0, qh, kh, vh, t0.positions, oh)
    torch.cuda.synchronize()
    od = lib.patch(0, 0, qs[0].cuda(), ks[0].cuda(), vs[0].cuda(), t0.positions)
    torch.cuda.synchronize()
    assert torch.equal(oh, od.cpu())
    # batched host-buffer call == batched device call
    qh, kh, vh = [x.cpu().contiguous().pin_memory() for x in (q, k, v)]
    oh = torch.empty_like(qh).pin_memory()
    lib.patch_batch_host([t.task_id for t in wl.tasks], [len(t.positions) for t in wl.tasks], 0, qh, kh, vh,
                         np.concatenate([t.positions for t in wl.tasks]), oh)
    torch.cuda.synchronize()
    assert torch.equal(oh, out.cpu())
    lib.close()


# ------------------------------------------------------------------------------------------------
# boundary behaviour through the C ABI (P13, P14)
# ------------------------------------------------------------------------------------------------
def test_p14_rejections_match_oracle_and_leave_state_unchanged():
    bnd = _binding()
    cfg = synth.GraftConfig("rej", 2, 4, 2, 64, 8, 1e4, 1, 10, 10, 0, 1, 1, 1, 0)
    wl = synth.make_workload(cfg, 1)
    wl.tasks[0].capacity = 64
    orc, lib, seg_ids = T.make_pair(cfg, wl, 1, n_pages=8, max_tasks=4)
    s0 = seg_ids[0]
    cases = [
        ({"task_id": 0, "entries": [(99, 0, 4, 0)]}, O.Plan(0, [O.PlanEntry(99, 0, 4, 0)])),
        ({"task_id": 0, "entries": [(s0, 8, 4, 0)]}, O.Plan(0, [O.PlanEntry(s0, 8, 4, 0)])),
        ({"task_id": 0, "entries": [(s0, -1, 4, 0)]}, O.Plan(0, [O.PlanEntry(s0, -1, 4, 0)])),
        ({"task_id": 0, "entries": [(s0, 0, 0, 0)]}, O.Plan(0, [O.PlanEntry(s0, 0, 0, 0)])),
        ({"task_id": 0, "entries": [(s0, 0, 4, -2)]}, O.Plan(0, [O.PlanEntry(s0, 0, 4, -2)])),
        ({"task_id": 0, "entries": [(s0, 0, 4, 0)], "capacity_tokens": 3}, O.Plan(0, [O.PlanEntry(s0, 0, 4, 0)], [], 3)),
        ({"task_id": 0, "entries": [(s0, 0, 4, 0), (s0, 4, 4, 3)]}, O.Plan(0, [O.PlanEntry(s0, 0, 4, 0), O.PlanEntry(s0, 4, 4, 3)])),
        ({"task_id": 0, "entries": [(s0, 0, 4, 0)], "holes": [(2, 4)]}, O.Plan(0, [O.PlanEntry(s0, 0, 4, 0)], [O.Hole(2, 4)])),
        ({"task_id": 0, "entries": [(s0, 0, 4, 0)], "capacity_tokens": 65}, O.Plan(0, [O.PlanEntry(s0, 0, 4, 0)], [], 65)),
        ({"task_id": 0, "entries": []}, O.Plan(0, [], [])),
        ({"task_id": -1, "entries": [(s0, 0, 4, 0)]}, O.Plan(-1, [O.PlanEntry(s0, 0, 4, 0)])),
        ({"task_id": 4, "entries": [(s0, 0, 4, 0)]}, O.Plan(4, [O.PlanEntry(s0, 0, 4, 0)])),
    ]
    for c_plan, o_plan in cases:
        with pytest.raises(O.OracleError) as eo:
            orc.stitch([o_plan])
        with pytest.raises(bnd.FcgError) as eg:
            lib.stitch([c_plan])
        assert eg.value.status == eo.value.status, (c_plan, eg.value, eo.value)
        info = lib.pool_info()
        assert info["n_pages_free"] == 8 and info["n_tasks_live"] == 0
    # pool exhaustion: 64 tokens = 8 pages fits, a second task does not; the batch rolls back as a whole
    good = {"task_id": 1, "entries": [(s0, 0, 10, 0)], "capacity_tokens": 64}
    with pytest.raises(bnd.FcgError) as eg:
        lib.stitch([good, {"task_id": 2, "entries": [(s0, 0, 4, 0)]}])
    assert eg.value.status == bnd.FCG_ERR_OUT_OF_PAGES and lib.pool_info()["n_tasks_live"] == 0
    with pytest.raises(bnd.FcgError) as eg:
        lib.stitch([good, good])
    assert eg.value.status == bnd.FCG_ERR_BAD_TASK
    lib.stitch([good])
    assert np.array_equal(lib.task_page_table_host(1), np.arange(8))
    with pytest.raises(bnd.FcgError) as eg:
        lib.stitch([good])
    assert eg.value.status == bnd.FCG_ERR_BAD_TASK
    # release order: pages come back so that the next task gets them in ascending logical order (R9)
    lib.task_release(1)
    orc.stitch([O.Plan(1, [O.PlanEntry(s0, 0, 10, 0)], [], 64)])
    orc.task_release(1)
    orc.stitch([O.Plan(2, [O.PlanEntry(s0, 0, 10, 0)], [], 24), O.Plan(3, [O.PlanEntry(s0, 0, 10, 0)], [], 17)])
    lib.stitch([{"task_id": 2, "entries": [(s0, 0, 10, 0)], "capacity_tokens": 24},
                {"task_id": 3, "entries": [(s0, 0, 10, 0)], "capacity_tokens": 17}])
    for tid in (2, 3):
        assert np.array_equal(lib.task_page_table_host(tid), np.asarray(orc.tasks[tid].page_table, np.int32))
    # device copy of the table == host copy (P13), ids unique across live tasks
    ids = []
    for tid in (2, 3):
        ptr, n_pages, _ = lib.task_page_table(tid)
        host = lib.task_page_table_host(tid)
        torch.cuda.synchronize()

        class _DevView:      # zero-copy view of the library's device table
            __cuda_array_interface__ = {"shape": (n_pages,), "typestr": "<i4", "data": (ptr, False), "version": 3}
        dev = torch.as_tensor(_DevView(), device="cuda")
        assert np.array_equal(dev.cpu().numpy(), host)
        ids += host.tolist()
    assert len(set(ids)) == len(ids) and max(ids) < 8
    # patch argument errors
    q, k, v = [x.cuda() for x in synth.patch_qkv(cfg, 2, 2, 1)]
    # (capacity of task 2 is 24: position 24 would append (R25) but 11..23 are unfilled; RANGE starts at max_task_tokens = 64)
    for pos, status in (([11, 10], bnd.FCG_ERR_INVALID_ARG), ([10, 64], bnd.FCG_ERR_RANGE), ([10, 24], bnd.FCG_ERR_UNFILLED),
                        ([12, 13], bnd.FCG_ERR_UNFILLED)):
        with pytest.raises(bnd.FcgError) as eg:
            lib.patch(2, 0, q, k, v, pos)
        assert eg.value.status == status
    with pytest.raises(bnd.FcgError) as eg:
        lib.patch(1, 0, q, k, v, [10, 11])
    assert eg.value.status == bnd.FCG_ERR_BAD_TASK
    with pytest.raises(bnd.FcgError) as eg:
        lib.segment_release(5)
    assert eg.value.status == bnd.FCG_ERR_BAD_SEGMENT
    lib.close()


def test_segment_release_reuses_ids_and_arena():
    cfg = synth.GraftConfig("segs", 1, 2, 2, 64, 16, 1e4, 4, 50, 50, 0, 1, 1, 1, 0)
    wl = synth.make_workload(cfg, 1)
    wl.tasks[0].capacity = 130
    orc, lib, seg_ids = T.make_pair(cfg, wl, 1, only_segments=[0, 1, 2, 3])
    free0 = lib.pool_info()["segments_bytes_free"]
    lib.segment_release(1)
    lib.segment_release(2)
    orc.segment_release(1)
    orc.segment_release(2)
    k, v = synth.segment_kv(cfg, 9, 100, 1)
    sid = lib.segment_register(k.cuda(), v.cuda(), 3)        # 100 tokens fit in the coalesced hole of 2 x 50
    assert sid == 1 == orc.segment_register(synth.to_bits(k), synth.to_bits(v), 3)
    assert lib.pool_info()["segments_bytes_free"] == free0
    # a strided (non-contiguous) source registers correctly
    big_k = torch.randn(1, 2, 77, 2, 64, device="cuda").to(torch.bfloat16)
    big_v = torch.randn(1, 2, 77, 2, 64, device="cuda").to(torch.bfloat16)
    ks, vs = big_k[:, :, 10:40, 1, :], big_v[:, :, 10:40, 1, :]
    lib.segment_release(3)
    orc.segment_release(3)
    sid2 = lib.segment_register(ks, vs, 0)
    assert sid2 == 2 == orc.segment_register(synth.to_bits(ks.contiguous()), synth.to_bits(vs.contiguous()), 0)
    lib.stitch([{"task_id": 0, "entries": [(sid2, 0, 30, 0), (sid, 0, 100, 30)]}])
    orc.stitch([O.Plan(0, [O.PlanEntry(sid2, 0, 30, 0), O.PlanEntry(sid, 0, 100, 30)])])
    wl.tasks[0].task_id = 0
    T.compare_stitched(orc, lib, wl)
    lib.close()


# ------------------------------------------------------------------------------------------------
# both attention kernels against the oracle on the same inputs (policy forced either way)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n,Hq,Hkv,ctx", [(64, 4, 4, 700), (16, 2, 2, 300), (48, 8, 2, 1000), (128, 4, 1, 2100), (3, 4, 2, 70)])
@pytest.mark.parametrize("tc_min_rows", [0, 2 ** 31 - 1])
def test_tcgen05_and_split_paths_match_oracle(n, Hq, Hkv, ctx, tc_min_rows):
    cfg = synth.GraftConfig("paths", 2, Hq, Hkv, 128, 16, 1e4, 3, ctx // 3, ctx // 3 + 40, 500, 1, 3, 3, 0,
                            holes=((0, max(1, n // 4)), (-1, n - max(1, n // 4))) if n > 1 else ((-1, 1),))
    wl = synth.make_workload(cfg, 13)
    orc, lib, seg_ids = T.make_pair(cfg, wl, 13)
    lib.set_attn_policy(tc_min_rows)
    c_plans, o_plans = T.plans_of(wl, seg_ids)
    orc.stitch(o_plans)
    lib.stitch(c_plans)
    out, ref = T.run_patch_both(orc, lib, cfg, wl.tasks[0], 14)
    assert lib.stats()["last_attn_path"] == (2 if tc_min_rows == 0 else 1)
    T.assert_attn_close(out, ref, f"path {'tc' if tc_min_rows == 0 else 'split'} n={n}")
    T.compare_cache_bits(orc, lib, 0, wl.tasks[0].positions)
    lib.close()


# ------------------------------------------------------------------------------------------------
# P11 split invariance with the split count FORCED, so that one CTA walks many more KV tiles than the
# shared-memory ring has stages (the auto choice gives small test grids many splits of a few tiles each
# and never exercises ring wrap-around); also the bench's launch shape (one split over the whole cache).
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n,Hq,Hkv,ctx", [(64, 2, 2, 4096), (20, 8, 2, 1500), (130, 2, 1, 2600)])
@pytest.mark.parametrize("tc_min_rows", [0, 2 ** 31 - 1])
@pytest.mark.parametrize("force_splits", [1, 2, 5])
def test_forced_split_counts_long_tile_loops(n, Hq, Hkv, ctx, tc_min_rows, force_splits):
    cfg = synth.GraftConfig("longloop", 1, Hq, Hkv, 128, 16, 1e4, 3, ctx // 3, ctx // 3 + 40, 500, 1, 3, 3, 0,
                            holes=((0, max(1, n // 4)), (-1, n - max(1, n // 4))))
    wl = synth.make_workload(cfg, 21)
    orc, lib, seg_ids = T.make_pair(cfg, wl, 21)
    lib.set_attn_policy(tc_min_rows, force_splits)
    c_plans, o_plans = T.plans_of(wl, seg_ids)
    orc.stitch(o_plans)
    lib.stitch(c_plans)
    out, ref = T.run_patch_both(orc, lib, cfg, wl.tasks[0], 22)
    st = lib.stats()
    assert st["last_attn_path"] == (2 if tc_min_rows == 0 else 1)
    assert st["last_attn_splits"] == force_splits
    T.assert_attn_close(out, ref, f"forced splits {force_splits}, path {st['last_attn_path']}, n={n}")
    lib.close()


# ------------------------------------------------------------------------------------------------
# tcgen05 path details: every page size (one TMA box per page and 64-column half), two 128-row Q tiles
# per CTA (R > 128), ragged last tiles, and a cache pool poisoned with NaN bit patterns (page slack and
# masked positions must never reach the output: DESIGN R10)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("P", [8, 16, 32, 64])
@pytest.mark.parametrize("n,Hq,Hkv,ctx", [(40, 4, 2, 1000), (70, 8, 2, 777), (260, 2, 2, 1500)])
def test_tcgen05_page_sizes_two_q_tiles_and_poisoned_pool(P, n, Hq, Hkv, ctx):
    cfg = synth.GraftConfig("tcpages", 2, Hq, Hkv, 128, P, 1e4, 3, ctx // 3, ctx // 3 + 40, 500, 1, 3, 3, 0,
                            holes=((0, max(1, n // 4)), (-1, n - max(1, n // 4))))
    wl = synth.make_workload(cfg, 31)
    orc, lib, seg_ids = T.make_pair(cfg, wl, 31)
    info = lib.pool_info()
    pool = lib.arena[info["k_pool_offset"]:info["v_pool_offset"] + info["pool_bytes"]]
    pool.fill_(0xFF)                                   # every bf16 in both pools is a NaN until written
    torch.cuda.synchronize()
    lib.set_attn_policy(0)
    c_plans, o_plans = T.plans_of(wl, seg_ids)
    orc.stitch(o_plans)
    lib.stitch(c_plans)
    out, ref = T.run_patch_both(orc, lib, cfg, wl.tasks[0], 32)
    assert lib.stats()["last_attn_path"] == 2
    assert torch.isfinite(out.float()).all()
    T.assert_attn_close(out, ref, f"tc P={P} n={n} G={Hq // Hkv}")
    # the same again with forced splits (partials + combine)
    lib.set_attn_policy(0, 3)
    out2 = lib.patch(0, 0, *[x.cuda().contiguous() for x in synth.patch_qkv(cfg, 0, len(wl.tasks[0].positions), 32, "cpu")],
                     wl.tasks[0].positions)
    torch.cuda.synchronize()
    T.assert_attn_close(out2, ref, f"tc P={P} n={n} 3 splits")
    lib.close()


@pytest.mark.parametrize("tc_min_rows", [0, 2 ** 31 - 1])
def test_growing_scores_force_the_rescale_path(tc_min_rows):
    """Scores that grow steadily along the cache (keys scaled by position, queries aligned with them) push the running
    row max up by far more than the lazy-rescale threshold (2^8) many times over: the O-rescale branch of every CTA
    class (prefill-like 2 Q tiles, tile-parity streams, row streams / decode) and of the split-KV kernel must run."""
    B = _binding()
    L, Hq, Hkv, D, T_ = 1, 4, 2, 128, 700
    cfg = synth.GraftConfig("grow", L, Hq, Hkv, D, 16, 1e4, 1, 8, 8, 0, 1, 1, 1, 0)
    wl = synth.make_workload(cfg, 1)
    wl.tasks[0].entries, wl.tasks[0].holes, wl.tasks[0].capacity = [], [(0, T_)], T_
    orc, lib, _ = T.make_pair(cfg, wl, 1, only_segments=[0], n_pages=T_ // 16 + 4)
    lib.set_attn_policy(tc_min_rows, 0)
    orc.stitch([O.Plan(0, [], [O.Hole(0, T_)], T_)])
    lib.stitch([{"task_id": 0, "entries": [], "holes": [(0, T_)], "capacity_tokens": T_}])
    g = torch.Generator().manual_seed(3)
    u = torch.rand(D, generator=g) + 0.5                                   # all-positive direction
    u = u / u.norm()
    ramp = torch.linspace(0.05, 1.0, T_)                                   # key length grows with the position
    k = (u[None, None, None, :] * ramp[None, :, None, None] * 30.0).expand(L, T_, Hkv, D).to(torch.bfloat16).contiguous()
    q = (u[None, None, None, :] * 25.0).expand(L, T_, Hq, D).to(torch.bfloat16).contiguous()   # s_x up to 25*30/sqrt(128) = 66
    v = torch.randn(L, T_, Hkv, D, generator=g).to(torch.bfloat16)
    pos = np.arange(T_, dtype=np.int32)
    ref = orc.patch(0, 0, synth.to_bits(q), synth.to_bits(k), synth.to_bits(v), pos)
    out = lib.patch(0, 0, q.cuda(), k.cuda(), v.cuda(), pos)
    torch.cuda.synchronize()
    T.assert_attn_close(out, ref, "prefill-like, growing scores")
    for n in (1, 20, 100):                                                 # re-patch the tail: the other CTA classes
        sl = slice(T_ - n, T_)
        ref = orc.patch(0, 0, synth.to_bits(q[:, sl]), synth.to_bits(k[:, sl]), synth.to_bits(v[:, sl]), pos[sl])
        out = lib.patch(0, 0, q[:, sl].contiguous().cuda(), k[:, sl].contiguous().cuda(), v[:, sl].contiguous().cuda(), pos[sl])
        torch.cuda.synchronize()
        T.assert_attn_close(out, ref, f"growing scores, last {n} tokens")
    lib.close()
