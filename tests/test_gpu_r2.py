"""Round-2 GPU parity tests of the host planner's new behaviour, all through the C ABI against the oracle:

* R25 appends beyond the reserved capacity: the hand-computed page-table script the oracle is pinned with
  (tests/golden/page_growth.txt) replayed on the C library; a 130-step decode past the stitched capacity;
* patch plans: 32 per-layer calls captured into ONE CUDA graph, replayed with new tensor contents;
* R29 stream ordering: tasks patched on different streams share the split-KV partials and the plan blobs;
* host / rope variants validate before they enqueue anything.
"""
import numpy as np
import pytest
import torch

import fcg_testlib as T
from oracle import fcg_oracle as O
from paper_2606_13097_b200 import synth
from test_oracle_pins_r2 import growth_script

pytestmark = pytest.mark.gpu


def _B():
    from paper_2606_13097_b200 import binding
    return binding


def _bits(rng, shape):
    x = torch.from_numpy(rng.standard_normal(shape).astype(np.float32)).to(torch.bfloat16)
    return x, synth.to_bits(x)


def test_growth_script_by_hand_on_the_c_library():
    B = _B()
    L, Hq, Hkv, D = 1, 2, 1, 64
    rng = np.random.default_rng(1)
    lib = B.FcgLibrary(n_layers=L, n_q_heads=Hq, n_kv_heads=Hkv, head_dim=D, page_size=8, max_segments=2, max_tasks=4,
                       max_task_tokens=32, n_pages=8, segment_tokens=64)
    # the script is written for P = 4 / max 16 tokens; the library's smallest page is 8 tokens: every token count x 2
    k, kb = _bits(rng, (L, Hkv, 12, D))
    v, vb = _bits(rng, (L, Hkv, 12, D))
    sid = lib.segment_register(k.cuda(), v.cuda(), 0)
    for op, args, status, table, cap, free in growth_script():
        got = B.FCG_OK
        try:
            if op == "stitch":
                t, c = args[0], 2 * args[1]
                lib.stitch([{"task_id": t, "entries": [(sid, 0, min(c, 12), 0)], "holes": [(12, c - 12)] if c > 12 else [],
                             "capacity_tokens": c}])
            elif op == "release":
                lib.task_release(args[0])
            else:
                t, pos = args[0], np.asarray([[2 * p, 2 * p + 1] for p in args[1:]], np.int32).ravel()
                q, _ = _bits(rng, (L, pos.size, Hq, D))
                kk, _ = _bits(rng, (L, pos.size, Hkv, D))
                lib.patch(t, 0, q.cuda(), kk.cuda(), kk.cuda(), pos)
        except B.FcgError as e:
            got = e.status
        what = f"{op} {args}"
        assert got == status, what
        assert lib.task_page_table_host(0).tolist() == table, what
        assert lib.pool_info()["n_pages_free"] == free, what
        assert lib.task_page_table(0)[1] == len(table)
    torch.cuda.synchronize()
    lib.close()


@pytest.mark.parametrize("D,Hq,Hkv", [(128, 8, 2), (64, 4, 4), (256, 4, 2), (96, 4, 2)])
def test_decode_130_steps_past_the_stitched_capacity(D, Hq, Hkv):
    """Eq. 6's x_mid is decoded token by token without reserving room for it (R25): stitch with capacity = T exactly,
    then 130 single-token patches, every one an append; 130 tokens at P = 16 cross 8 page boundaries.  A second task
    grows in between so that the pages interleave.  Every step's output, the final page tables and the cache bits are
    compared with the oracle."""
    L, P = 2, 16
    cfg = synth.GraftConfig("grow", L, Hq, Hkv, D, P, 1e4, 3, 40, 90, 500, 2, 2, 2, 0)
    wl = synth.make_workload(cfg, 5)
    orc, lib, seg_ids = T.make_pair(cfg, wl, 5, n_pages=64, max_task_tokens=512)
    c_plans, o_plans = T.plans_of(wl, seg_ids)
    for cp, op in zip(c_plans, o_plans):
        cp["capacity_tokens"] = 0
        op.capacity_tokens = 0
    orc.stitch(o_plans)
    lib.stitch(c_plans)
    rng = np.random.default_rng(9)
    ends = [orc.tasks[t.task_id].capacity for t in wl.tasks]
    worst = 0.0
    for step in range(130):
        for ti in ((0, 1) if step % 3 == 0 else (0,)):           # task 1 grows every third step
            pos = np.asarray([ends[ti]], np.int32)
            q, qb = _bits(rng, (L, 1, Hq, D))
            k, kb = _bits(rng, (L, 1, Hkv, D))
            v, vb = _bits(rng, (L, 1, Hkv, D))
            ref = orc.patch(ti, 0, qb, kb, vb, pos)
            out = lib.patch(ti, 0, q.cuda(), k.cuda(), v.cuda(), pos)
            worst = max(worst, T.assert_attn_close(out, ref, f"step {step} task {ti}"))
            ends[ti] += 1
    assert len(orc.tasks[0].page_table) - (-(-(ends[0] - 130) // P)) >= 8
    for t in wl.tasks:
        ot = orc.tasks[t.task_id]
        assert np.array_equal(lib.task_page_table_host(t.task_id), np.asarray(ot.page_table, np.int32))
        assert lib.task_page_table(t.task_id)[2] == ot.n_tokens == ends[t.task_id]
        for layer in range(L):
            kg, vg = lib.task_read(t.task_id, layer, 0, ot.capacity)
            f = ot.filled
            assert f.all()
            assert np.array_equal(synth.to_bits(vg)[:, f], ot.v[layer][:, f])
            T.assert_k_within_1ulp(synth.to_bits(kg)[:, f], ot.k[layer][:, f], f"task {t.task_id} layer {layer}")
    assert lib.pool_info()["n_pages_free"] == orc.pool.available()
    # growth is refused at max_task_tokens and when the pool is empty, with nothing changed
    B = _B()
    q, _ = _bits(rng, (L, 1, Hq, D))
    k, _ = _bits(rng, (L, 1, Hkv, D))
    with pytest.raises(B.FcgError) as e:
        lib.patch(0, 0, q.cuda(), k.cuda(), k.cuda(), [512])
    assert e.value.status == B.FCG_ERR_RANGE
    with pytest.raises(B.FcgError) as e:
        lib.patch(0, 0, q.cuda(), k.cuda(), k.cuda(), [ends[0] + 1])          # a gap is a hole, not an append
    assert e.value.status == B.FCG_ERR_UNFILLED
    assert lib.task_page_table(0)[2] == ends[0]
    lib.close()


def test_task_shift_beyond_capacity_grows_like_the_oracle():
    L, Hq, Hkv, D, P = 2, 4, 2, 128, 16
    cfg = synth.GraftConfig("growshift", L, Hq, Hkv, D, P, 1e4, 2, 70, 70, 100, 1, 1, 1, 0)
    wl = synth.make_workload(cfg, 3)
    orc, lib, seg_ids = T.make_pair(cfg, wl, 3, n_pages=40, max_task_tokens=400)
    c_plans, o_plans = T.plans_of(wl, seg_ids)
    c_plans[0]["capacity_tokens"] = 0
    o_plans[0].capacity_tokens = 0
    orc.stitch(o_plans)
    lib.stitch(c_plans)
    cap = orc.tasks[0].capacity
    for args in ((0, 30, 20, cap + 40), (0, 0, 25, cap - 5), (0, cap + 40, 20, cap + 45)):
        orc.task_shift(*args)
        lib.task_shift(*args)
        ot = orc.tasks[0]
        assert np.array_equal(lib.task_page_table_host(0), np.asarray(ot.page_table, np.int32)), args
        assert lib.pool_info()["n_pages_free"] == orc.pool.available()
        for layer in range(L):
            kg, vg = lib.task_read(0, layer, 0, ot.capacity)
            f = ot.filled
            assert np.array_equal(synth.to_bits(vg)[:, f], ot.v[layer][:, f]), args
            T.assert_k_within_1ulp(synth.to_bits(kg)[:, f], ot.k[layer][:, f], f"shift {args}")
    B = _B()
    with pytest.raises(B.FcgError) as e:
        lib.task_shift(0, cap + 45, 20, 390)
    assert e.value.status == B.FCG_ERR_RANGE
    lib.close()


def test_patch_plan_captured_into_one_cuda_graph_and_replayed():
    """The per-layer call pattern of a real model as pure launches: a plan, 32 per-layer fcg_patch_planned calls captured
    into one CUDA graph, the graph replayed twice with new q / k / v contents -- each replay against the oracle."""
    B = _B()
    L, Hq, Hkv, D, P = 32, 4, 4, 128, 16
    cfg = synth.GraftConfig("plan", L, Hq, Hkv, D, P, 1e4, 3, 300, 500, 2000, 1, 3, 3, 0, holes=((0, 16), (-1, 24)))
    wl = synth.make_workload(cfg, 2)
    orc, lib, seg_ids = T.make_pair(cfg, wl, 2)
    c_plans, o_plans = T.plans_of(wl, seg_ids)
    orc.stitch(o_plans)
    lib.stitch(c_plans)
    task = wl.tasks[0]
    n = len(task.positions)
    # an unplanned call refuses to be captured (it would bake a host blob into the graph)
    q0, k0, v0 = [x.cuda() for x in synth.patch_qkv(cfg, 0, n, 1)]
    out = torch.empty_like(q0)
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    plan = lib.patch_plan_create([0], [n], task.positions, 1)
    assert lib.pool_info()["n_segments_live"] == len(seg_ids)
    lib.patch_planned(plan, 0, q0[:1], k0[:1], v0[:1], out[:1])       # warm-up outside the capture (first-launch setup)
    torch.cuda.synchronize()
    side.wait_stream(torch.cuda.current_stream())
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=side):
        with pytest.raises(B.FcgError) as e:
            lib.patch(0, 0, q0[:1], k0[:1], v0[:1], task.positions, out[:1])
        assert e.value.status == B.FCG_ERR_INVALID_ARG
        for layer in range(L):
            lib.patch_planned(plan, layer, q0[layer:layer + 1], k0[layer:layer + 1], v0[layer:layer + 1], out[layer:layer + 1])
    torch.cuda.synchronize()
    s0 = lib.stats()
    for rep, seed in enumerate((11, 12)):
        q, k, v = synth.patch_qkv(cfg, 0, n, seed)
        q0.copy_(q.cuda()), k0.copy_(k.cuda()), v0.copy_(v.cuda())
        out.zero_()
        torch.cuda.synchronize()
        g.replay()
        torch.cuda.synchronize()
        ref = orc.patch(0, 0, synth.to_bits(q), synth.to_bits(k), synth.to_bits(v), task.positions)
        T.assert_attn_close(out, ref, f"graph replay {rep}")
        T.compare_cache_bits(orc, lib, 0, task.positions)
    assert lib.stats()["scatter_launches"] == s0["scatter_launches"]          # replays make no library calls
    # the same plan outside a graph, several layers per call
    q, k, v = synth.patch_qkv(cfg, 0, n, 13)
    out2 = lib.patch_planned(plan, 4, q[4:12].cuda().contiguous(), k[4:12].cuda().contiguous(), v[4:12].cuda().contiguous(),
                             torch.empty_like(q[4:12]).cuda())
    torch.cuda.synchronize()
    ref = orc.patch(0, 4, synth.to_bits(q[4:12]), synth.to_bits(k[4:12]), synth.to_bits(v[4:12]), task.positions)
    T.assert_attn_close(out2, ref, "planned call of 8 layers")
    # a plan dies with its task
    lib.task_release(0)
    with pytest.raises(B.FcgError) as e:
        lib.patch_planned(plan, 0, q0[:1], k0[:1], v0[:1], out[:1])
    assert e.value.status == B.FCG_ERR_BAD_TASK
    free0 = lib.pool_info()["segments_bytes_free"]
    lib.patch_plan_destroy(plan)
    assert lib.pool_info()["segments_bytes_free"] > free0
    lib.close()


def test_plan_with_forced_splits_and_growth_matches_oracle():
    """plan creation does the growth (R25) and the split choice; planned calls with split-KV partials + combine."""
    L, Hq, Hkv, D, P = 4, 8, 2, 128, 16
    cfg = synth.GraftConfig("plangrow", L, Hq, Hkv, D, P, 5e5, 2, 700, 900, 4000, 1, 2, 2, 0)
    wl = synth.make_workload(cfg, 4)
    orc, lib, seg_ids = T.make_pair(cfg, wl, 4, n_pages=200, max_task_tokens=2500)
    c_plans, o_plans = T.plans_of(wl, seg_ids)
    c_plans[0]["capacity_tokens"] = 0
    o_plans[0].capacity_tokens = 0
    orc.stitch(o_plans)
    lib.stitch(c_plans)
    cap = orc.tasks[0].capacity
    pos = np.arange(cap, cap + 40, dtype=np.int32)
    lib.set_attn_policy(1, 3)
    plan = lib.patch_plan_create([0], [40], pos, 2)
    assert lib.task_page_table(0)[1] == -(-(cap + 40) // P)
    q, k, v = synth.patch_qkv(cfg, 0, 40, 6)
    out = torch.empty_like(q).cuda()
    for lb in (0, 2):
        lib.patch_planned(plan, lb, q[lb:lb + 2].cuda().contiguous(), k[lb:lb + 2].cuda().contiguous(),
                          v[lb:lb + 2].cuda().contiguous(), out[lb:lb + 2])
    torch.cuda.synchronize()
    assert lib.stats()["last_attn_splits"] == 3
    ref = orc.patch(0, 0, synth.to_bits(q), synth.to_bits(k), synth.to_bits(v), pos)
    T.assert_attn_close(out, ref, "planned, 3 splits, grown task")
    assert np.array_equal(lib.task_page_table_host(0), np.asarray(orc.tasks[0].page_table, np.int32))
    lib.patch_plan_destroy(plan)
    lib.close()


def test_two_streams_share_scratch_and_pages_safely():
    """R29: two tasks patched alternately on two streams with KV splits forced (both use the partials at the start of
    the scratch area and cycle through the same plan blobs); one task is released and re-stitched on the other
    stream while its attention may still be running.  Every result must match the oracle."""
    L, Hq, Hkv, D, P = 4, 8, 2, 128, 16
    cfg = synth.GraftConfig("streams", L, Hq, Hkv, D, P, 1e4, 4, 600, 900, 3000, 2, 2, 3, 0, holes=((-1, 24),))
    wl = synth.make_workload(cfg, 7)
    orc, lib, seg_ids = T.make_pair(cfg, wl, 7, n_pages=2 * 200)
    c_plans, o_plans = T.plans_of(wl, seg_ids)
    orc.stitch(o_plans)
    lib.set_attn_policy(1, 4)
    s = [torch.cuda.Stream(), torch.cuda.Stream()]
    torch.cuda.synchronize()
    lib.stitch(c_plans, stream=s[0])
    outs, refs = [], []
    for it in range(6):
        for ti, t in enumerate(wl.tasks):
            st = s[(it + ti) % 2]
            q, k, v = synth.patch_qkv(cfg, t.task_id, len(t.positions), 100 + it)
            with torch.cuda.stream(st):
                qd, kd, vd = q.cuda(non_blocking=True), k.cuda(non_blocking=True), v.cuda(non_blocking=True)
                outs.append((lib.patch(t.task_id, 0, qd, kd, vd, t.positions, stream=st), qd, kd, vd))
            refs.append(orc.patch(t.task_id, 0, synth.to_bits(q), synth.to_bits(k), synth.to_bits(v), t.positions))
        if it == 2:
            # task 1 goes away and comes back (same pages, LIFO) on the OTHER stream than its last patch ran on
            other = s[(it + 1 + 1) % 2]
            lib.task_release(1)
            orc.task_release(1)
            lib.stitch([c_plans[1]], stream=other)
            orc.stitch([o_plans[1]])
    torch.cuda.synchronize()
    for i, ((out, *_), ref) in enumerate(zip(outs, refs)):
        T.assert_attn_close(out, ref, f"call {i}")
    lib.close()


def test_host_and_rope_variants_validate_before_enqueueing():
    B = _B()
    cfg = synth.scaled(synth.C1, holes=((1, 32), (-1, 32)))
    wl = synth.make_workload(cfg, 2)
    orc, lib, seg_ids = T.make_pair(cfg, wl, 2)
    c_plans, o_plans = T.plans_of(wl, seg_ids)
    orc.stitch(o_plans)
    lib.stitch(c_plans)
    task = wl.tasks[0]
    mid = np.arange(task.holes[0][0], task.holes[0][0] + 32, dtype=np.int32)
    end = np.arange(task.holes[1][0], task.holes[1][0] + 32, dtype=np.int32)
    q, k, v = synth.patch_qkv(cfg, 0, 32, 9)
    qh, kh, vh = [x.contiguous().pin_memory() for x in (q, k, v)]
    oh = torch.empty_like(qh).pin_memory()
    s0 = lib.stats()
    for fn, args in ((lib.patch_host, (0, 0, qh, kh, vh, end, oh)), (lib.patch_rope, (0, 0, q.cuda(), k.cuda(), v.cuda(), end))):
        with pytest.raises(B.FcgError) as e:              # the end patch would attend over the unfilled mid hole
            fn(*args)
        assert e.value.status == B.FCG_ERR_UNFILLED
    s1 = lib.stats()
    assert all(s1[f] == s0[f] for f in s1 if f.endswith("_launches")), "a rejected call launched something"
    ref = orc.patch(0, 0, synth.to_bits(q), synth.to_bits(k), synth.to_bits(v), mid)
    lib.patch_host(0, 0, qh, kh, vh, mid, oh)
    torch.cuda.synchronize()
    T.assert_attn_close(oh, ref, "host patch after the rejections")
    lib.close()


def test_stitch_prefetch_overlaps_and_matches_the_oracle():
    """NEXT-3: offloaded segments (one of them fp8) named by a plan come back through the copy engine while the resident
    entries are stitched; same cache, same page tables, the segments end up resident.  Then the no-room case: a segment
    that finds no arena range stays offloaded and is read in place."""
    L, Hq, Hkv, D, P = 4, 4, 2, 128, 16
    from paper_2606_13097_b200.binding import FcgLibrary
    rng = np.random.default_rng(21)
    lens = [400, 250, 600, 130]
    lib = FcgLibrary(n_layers=L, n_q_heads=Hq, n_kv_heads=Hkv, head_dim=D, page_size=P, rope_base=1e4, max_segments=12, max_tasks=3,
                     max_task_tokens=2048, n_pages=300, segment_tokens=sum(lens) + 40, host_tier_tokens=1200)
    orc = O.OracleLibrary(L, Hq, Hkv, D, page_size=P, rope_base=1e4, n_pages=300, max_task_tokens=2048)
    for i, n in enumerate(lens):
        k, kb = _bits(rng, (L, Hkv, n, D))
        v, vb = _bits(rng, (L, Hkv, n, D))
        if i == 2:
            assert lib.segment_register_fp8(k.cuda(), v.cuda(), 100 * i) == orc.segment_register_fp8(kb, vb, 100 * i) == i
        else:
            assert lib.segment_register(k.cuda(), v.cuda(), 100 * i) == orc.segment_register(kb, vb, 100 * i) == i
    for sid in (0, 2):
        lib.segment_offload(sid)
        orc.segment_offload(sid)
    entries = [(0, 10, 380, 0), (1, 0, 250, 380), (2, 0, 600, 630), (3, 5, 100, 1230), (0, 0, 64, 1330)]
    plan = {"task_id": 0, "entries": entries, "holes": [], "capacity_tokens": 0}
    lib.stitch_prefetch([plan])
    orc.stitch([O.Plan(0, [O.PlanEntry(*e) for e in entries])], prefetch=True)
    torch.cuda.synchronize()

    def check(tid, what):
        ot = orc.tasks[tid]
        assert np.array_equal(lib.task_page_table_host(tid), np.asarray(ot.page_table, np.int32)), what
        for layer in range(L):
            kg, vg = lib.task_read(tid, layer, 0, ot.capacity)
            f = ot.filled
            assert np.array_equal(synth.to_bits(vg)[:, f], ot.v[layer][:, f]), what
            T.assert_k_within_1ulp(synth.to_bits(kg)[:, f], ot.k[layer][:, f], what)

    check(0, "stitch_prefetch")
    assert [lib.segment_info(i)[2] for i in range(4)] == [orc.segment_info(i)[2] for i in range(4)] == [True] * 4
    assert lib.stats()["prefetch_copies"] == 2
    # no room on the device tier: fill the arena, offload one segment, and ask for it again -- it is read in place
    lib.segment_offload(1)
    orc.segment_offload(1)
    filler, _ = _bits(rng, (L, Hkv, 100, D))
    B = _B()
    fillers = []
    while True:                                       # 100-token fillers until none fits: no free range of 250 tokens is left
        try:
            fillers.append(lib.segment_register(filler.cuda(), filler.cuda(), 0))
        except B.FcgError as e:
            assert e.status == B.FCG_ERR_OUT_OF_ARENA
            break
    assert 1 <= len(fillers) <= 6
    for _ in fillers:
        orc.segment_register(synth.to_bits(filler), synth.to_bits(filler), 0)
    lib.stitch_prefetch([{"task_id": 1, "entries": [(1, 0, 250, 0), (3, 0, 130, 250)], "holes": [], "capacity_tokens": 0}])
    orc.stitch([O.Plan(1, [O.PlanEntry(1, 0, 250, 0), O.PlanEntry(3, 0, 130, 250)])])
    torch.cuda.synchronize()
    check(1, "stitch_prefetch without room")
    assert lib.segment_info(1)[2] is False and lib.stats()["prefetch_copies"] == 2
    for fid in fillers:
        lib.segment_release(fid)
    lib.close()


@pytest.mark.parametrize("n,Hq,Hkv,ctx,P,splits", [(130, 2, 1, 2600, 16, 0), (260, 2, 2, 1500, 8, 2), (45, 8, 2, 1000, 64, 0), (300, 2, 2, 777, 16, 3),
                                                  (64, 16, 4, 4096, 32, 0), (200, 4, 4, 100, 16, 0)])
def test_cta_pair_kernel_matches_the_oracle(n, Hq, Hkv, ctx, P, splits):
    """the cta_group::2 variant of the > 128-rows class (fcg_set_attn_pairs): page sizes, ragged last tiles, a trailing row
    group whose second CTA holds no row, KV splits + combine, a mid hole and an appended patch -- all against the oracle,
    pool poisoned with NaN."""
    L, D = 2, 128
    cfg = synth.GraftConfig("pair", L, Hq, Hkv, D, P, 1e4, 2, ctx, ctx, 1000, 1, 1, 1, 0, holes=((-1, n),))
    wl = synth.make_workload(cfg, n + ctx)
    orc, lib, seg_ids = T.make_pair(cfg, wl, 3, n_pages=-(-(ctx + 2 * n + 8) // P) + 4, max_task_tokens=ctx + 2 * n + 8, workspace_bytes=128 << 20)
    info = lib.pool_info()
    lib.arena[info["k_pool_offset"]: info["k_pool_offset"] + 2 * info["pool_bytes"]].view(torch.int16).fill_(0x7FC1)
    c_plans, o_plans = T.plans_of(wl, seg_ids)
    orc.stitch(o_plans)
    lib.stitch(c_plans)
    lib.set_attn_pairs(True)
    lib.set_attn_policy(1, splits)
    task = wl.tasks[0]
    out, ref = T.run_patch_both(orc, lib, cfg, task, 5)
    assert lib.stats()["last_attn_path"] == 2
    T.assert_attn_close(out, ref, "pair kernel, patch at the end")
    T.compare_cache_bits(orc, lib, 0, task.positions)
    # a second, appended patch (grows the task): queries see the first patch too
    pos = np.arange(task.capacity, task.capacity + n, dtype=np.int32)
    out, ref = T.run_patch_both(orc, lib, cfg, task, 6, positions=pos)
    T.assert_attn_close(out, ref, "pair kernel, appended patch")
    # and the single-CTA kernel gives the same answer within the tolerance of both
    lib.set_attn_pairs(False)
    out2, ref2 = T.run_patch_both(orc, lib, cfg, task, 6, positions=pos)
    T.assert_attn_close(out2, ref2, "single-CTA kernel, same patch")
    assert float((out.float() - out2.float()).abs().max()) < 2e-2
    lib.close()


def test_mixed_class_batch_in_one_launch_matches_the_per_class_launches_and_the_oracle():
    """fcg_set_attn_mixed: a batch whose tasks fall into all three CTA classes (16, 30 and 50 tokens at G = 4: 64, 120 and
    200 rows per kv head) as ONE interleaved launch; with and without KV splits; against the oracle and against the default
    one-launch-per-class path (bit-identical: the same CTA program runs either way)."""
    L, Hq, Hkv, D, P = 3, 8, 2, 128, 16
    cfg = synth.GraftConfig("mixed", L, Hq, Hkv, D, P, 1e4, 4, 300, 900, 3000, 5, 2, 3, 0, total_min=500, total_max=2500,
                            distinct_segments=False, holes=((-1, 0),), patch_min=10, patch_max=60)
    wl = synth.make_workload(cfg, 8)
    for t, n in zip(wl.tasks, (16, 30, 50, 8, 64)):              # pin the patch sizes: rows 64, 120, 200, 32, 256
        b = t.holes[-1][0]
        t.holes[-1] = (b, n)
        t.capacity = b + n
        t.positions = np.arange(b, b + n, dtype=np.int32)
    orc, lib, seg_ids = T.make_pair(cfg, wl, 8, workspace_bytes=128 << 20)
    c_plans, o_plans = T.plans_of(wl, seg_ids)
    orc.stitch(o_plans)
    lib.stitch(c_plans)
    ids = [t.task_id for t in wl.tasks]
    npt = [len(t.positions) for t in wl.tasks]
    pos = np.concatenate([t.positions for t in wl.tasks]).astype(np.int32)
    qs = [synth.patch_qkv(cfg, t.task_id, len(t.positions), 3) for t in wl.tasks]
    q, k, v = [torch.cat([x[j] for x in qs], dim=1).contiguous() for j in range(3)]
    ref = np.concatenate([orc.patch(t.task_id, 0, synth.to_bits(x[0]), synth.to_bits(x[1]), synth.to_bits(x[2]), t.positions)
                          for t, x in zip(wl.tasks, qs)], axis=1)
    for splits in (0, 2):
        outs = []
        for mixed in (True, False):
            lib.set_attn_mixed(mixed)
            lib.set_attn_policy(1, splits)
            s0 = lib.stats()["attn_tc_launches"]
            outs.append(lib.patch_batch(ids, npt, 0, q.cuda(), k.cuda(), v.cuda(), pos))
            torch.cuda.synchronize()
            assert lib.stats()["attn_tc_launches"] - s0 == (1 if mixed else 3)
            T.assert_attn_close(outs[-1], ref, f"mixed={mixed} splits={splits}")
        assert torch.equal(outs[0], outs[1])
    lib.close()


def test_batches_beyond_the_launch_limit_are_rejected_before_anything_runs():
    """n_layers x n_tasks > 65535 would not fit the attention grid's z extent: INVALID_ARG, nothing launched (fcg.h)."""
    B = _B()
    lib = B.FcgLibrary(n_layers=2, n_q_heads=2, n_kv_heads=2, head_dim=64, page_size=16, rope_base=1e4, max_segments=1, max_tasks=4,
                       max_task_tokens=64, n_pages=8, segment_tokens=64)
    n_tasks = 40000
    q = torch.zeros((2, n_tasks, 2, 64), dtype=torch.bfloat16, device="cuda")
    before = lib.stats()
    with pytest.raises(B.FcgError) as e:
        lib.patch_batch(np.arange(n_tasks, dtype=np.int32), np.ones(n_tasks, np.int32), 0, q, q, q, np.zeros(n_tasks, np.int32))
    assert e.value.status == B.FCG_ERR_INVALID_ARG
    assert lib.stats() == before
    lib.close()
