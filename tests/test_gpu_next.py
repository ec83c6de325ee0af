"""GPU parity for the NEXT rows of SURVEY.md 8(f): interleaved RoPE pairs, the suffix re-graft of a
length-changing patch (fcg_task_shift), segment extraction (fcg_segment_extract) and single-token decode
attention.  Same bars as test_gpu_parity.py: page tables, V and copies bit-exact; rotated K within 1 bf16 ulp of
the oracle for every element; attention within 2e-2 relative + 1e-2 absolute."""
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


def _pair(cfg, seed=1, rope_mode=1, extra_pages=64, tweak=None, **kw):
    """oracle + CUDA library over the same workload; `tweak(wl)` edits the plans before capacities are sized."""
    wl = synth.make_workload(cfg, seed)
    if tweak is not None:
        tweak(wl)
    total_pages = sum(-(-t.capacity // cfg.page_size) for t in wl.tasks)
    orc, lib, seg_ids = T.make_pair(cfg, wl, seed, rope_mode=rope_mode, n_pages=total_pages + extra_pages,
                                    only_segments=list(range(cfg.n_segments)), **kw)
    return wl, orc, lib, seg_ids


def _grow(extra):
    def tweak(wl):
        for t in wl.tasks:
            t.capacity += extra
            t.holes = []
    return tweak


def _compare_task(orc, lib, task_id, what):
    """page table, token count, and every FILLED position of every layer: V bits, K within 1 ulp."""
    ot = orc.tasks[task_id]
    assert np.array_equal(lib.task_page_table_host(task_id), np.asarray(ot.page_table, np.int32)), f"{what}: page table"
    _, n_pages, n_tokens = lib.task_page_table(task_id)
    assert n_pages == len(ot.page_table) and n_tokens == ot.n_tokens, f"{what}: page / token count"
    hist = np.zeros(4, np.int64)
    for layer in range(orc.L):
        k, v = lib.task_read(task_id, layer, 0, ot.capacity)
        kb, vb = synth.to_bits(k), synth.to_bits(v)
        f = ot.filled
        assert np.array_equal(vb[:, f], ot.v[layer][:, f]), f"{what}: V not bit-exact (layer {layer})"
        hist += T.assert_k_within_1ulp(kb[:, f], ot.k[layer][:, f], f"{what} layer {layer}")
    return hist


# ------------------------------------------------------------------------------------------------
# NEXT-4: interleaved pairs
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("D", [64, 128, 256, 96, 192, 48])
def test_interleaved_rope_stitch(D):
    cfg = synth.GraftConfig("il", 2, 4, 2, D, 16, 1e4, 6, 40, 200, 3000, 1, 4, 4, 0)
    wl, orc, lib, seg_ids = _pair(cfg, seed=2, rope_mode=O.ROPE_INTERLEAVED)
    c_plans, o_plans = T.plans_of(wl, seg_ids)
    orc.stitch(o_plans)
    lib.stitch(c_plans)
    hist = T.compare_stitched(orc, lib, wl)
    assert hist[0] > 0.99 * hist.sum()
    # the interleaved result is NOT the half-split result (the flag does something)
    orc_h = O.OracleLibrary(cfg.n_layers, cfg.n_q_heads, cfg.n_kv_heads, D, page_size=16, rope_mode=1, rope_base=1e4)
    for s in range(cfg.n_segments):
        k, v = synth.segment_kv(cfg, s, int(wl.seg_lens[s]), 2, "cpu")
        orc_h.segment_register(synth.to_bits(k), synth.to_bits(v), int(wl.orig_starts[s]))
    orc_h.stitch(o_plans)
    f = orc.tasks[0].filled
    assert not np.array_equal(orc_h.tasks[0].k[:, :, f], orc.tasks[0].k[:, :, f])
    lib.close()


# ------------------------------------------------------------------------------------------------
# NEXT-1: length-changing patch = shift of the kept suffix, then the patch itself
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("rope_mode", [1, 2, 0])
@pytest.mark.parametrize("dlen", [5, -3, 16, -16, 37])
def test_task_shift_matches_oracle(rope_mode, dlen):
    cfg = synth.GraftConfig("shift", 2, 4, 2, 128, 16, 1e4, 5, 60, 150, 2000, 1, 3, 3, 0)
    wl, orc, lib, seg_ids = _pair(cfg, seed=3, rope_mode=rope_mode, tweak=_grow(64))
    task = wl.tasks[0]
    c_plans, o_plans = T.plans_of(wl, seg_ids)
    orc.stitch(o_plans)
    lib.stitch(c_plans)
    T_end = orc.tasks[0].n_tokens
    mid = T_end // 2 + 3                       # suffix [mid, T_end) moves by dlen (x_mid grew or shrank)
    orc.task_shift(0, mid, T_end - mid, mid + dlen)
    lib.task_shift(0, mid, T_end - mid, mid + dlen)
    _compare_task(orc, lib, 0, f"shift {dlen:+d}")
    if dlen > 0:
        # Eq. 6: the longer x_mid is patched into the gap; its queries see prefix + themselves
        pos = np.arange(mid, mid + dlen, dtype=np.int32)
        out, ref = T.run_patch_both(orc, lib, cfg, task, 3, positions=pos)
        T.assert_attn_close(out, ref, "patch into the widened hole")
        _compare_task(orc, lib, 0, "after the patch")
        # and a token appended after the moved suffix attends over prefix + x_mid + re-grafted suffix
        pos = np.asarray([T_end + dlen], np.int32)
        out, ref = T.run_patch_both(orc, lib, cfg, task, 4, positions=pos)
        T.assert_attn_close(out, ref, "decode step after the re-graft")
    lib.close()


def test_task_shift_rejections_and_page_recycling():
    B = _binding()
    cfg = synth.GraftConfig("shiftrej", 1, 2, 2, 64, 16, 1e4, 2, 64, 64, 100, 1, 1, 1, 0)
    wl = synth.make_workload(cfg, 1)
    wl.tasks[0].entries = [(0, 0, 64, 0)]
    wl.tasks[0].holes = []
    wl.tasks[0].capacity = 128
    orc, lib, seg_ids = T.make_pair(cfg, wl, 1, n_pages=11, only_segments=[0, 1])
    c_plans, o_plans = T.plans_of(wl, seg_ids)
    orc.stitch(o_plans)
    lib.stitch(c_plans)                                           # 8 pages used, 3 free
    for args, status in (((0, 64, 8, 0), B.FCG_ERR_UNFILLED), ((0, 32, 32, 100), B.FCG_ERR_RANGE),
                         ((0, -1, 4, 0), B.FCG_ERR_RANGE), ((0, 0, 0, 4), B.FCG_ERR_RANGE),
                         ((5, 0, 4, 4), B.FCG_ERR_BAD_TASK), ((0, 0, 64, 8), B.FCG_ERR_OUT_OF_PAGES)):
        with pytest.raises(B.FcgError) as e:
            lib.task_shift(*args)
        assert e.value.status == status, args
        with pytest.raises(O.OracleError) as eo:
            orc.task_shift(*args)
        assert eo.value.status == status, args
        assert lib.pool_info()["n_pages_free"] == orc.pool.available() == 3
    _compare_task(orc, lib, 0, "after rejections")
    for args in ((0, 40, 24, 50), (0, 50, 24, 41), (0, 0, 30, 90), (0, 30, 8, 30)):       # pages recycle through the pool
        orc.task_shift(*args)
        lib.task_shift(*args)
        _compare_task(orc, lib, 0, f"shift {args}")
        assert lib.pool_info()["n_pages_free"] == orc.pool.available()
    lib.close()


# ------------------------------------------------------------------------------------------------
# NEXT-2: segment extraction, and re-use of the extracted segment by another task
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("rope_mode", [1, 2])
def test_segment_extract_and_regraft(rope_mode):
    B = _binding()
    cfg = synth.GraftConfig("extract", 2, 4, 2, 128, 16, 5e5, 4, 50, 120, 4000, 1, 3, 3, 0)
    def drop_segment_3(wl):
        t, cursor, ents = wl.tasks[0], 0, []
        for (s_, b_, n_, _) in t.entries:
            if s_ != 3:
                ents.append((s_, b_, n_, cursor))
                cursor += n_
        t.entries, t.holes, t.capacity = ents, [], cursor

    wl, orc, lib, seg_ids = _pair(cfg, seed=2, rope_mode=rope_mode, tweak=drop_segment_3, max_tasks=3)
    # room for the extracted segments: the test library sizes its arena for the registered ones only
    lib.segment_release(3), orc.segment_release(3)
    c_plans, o_plans = T.plans_of(wl, seg_ids)
    orc.stitch(o_plans)
    lib.stitch(c_plans)
    filled = np.flatnonzero(orc.tasks[0].filled)
    b = int(filled[0]) + 7
    n = min(45, int(wl.seg_lens[3]))                             # fits the arena range freed above
    for new_start in (b, 0):
        so = orc.segment_extract(0, b, n, new_start)
        sg = lib.segment_extract(0, b, n, new_start)
        assert so == sg
        # stitch the new segment into a fresh task at another offset and compare caches
        tid = 1 if new_start == b else 2
        plan_c = {"task_id": tid, "entries": [(sg, 2, n - 2, 19)], "holes": [(0, 19)], "capacity_tokens": 19 + n}
        orc.stitch([O.Plan(tid, [O.PlanEntry(so, 2, n - 2, 19)], [O.Hole(0, 19)], 19 + n)])
        lib.stitch([plan_c])
        _compare_task(orc, lib, tid, f"graft of the extracted segment (orig_start {new_start})")
        lib.segment_release(sg), orc.segment_release(so)
    for args, status in (((0, int(filled[-1]), 4, 0), B.FCG_ERR_UNFILLED if int(filled[-1]) + 4 <= orc.tasks[0].capacity else B.FCG_ERR_RANGE),
                         ((0, b, n, -1), B.FCG_ERR_INVALID_ARG), ((7, b, n, 0), B.FCG_ERR_BAD_TASK),
                         ((0, b, 10 ** 6, 0), B.FCG_ERR_RANGE)):
        with pytest.raises(B.FcgError) as e:
            lib.segment_extract(*args)
        assert e.value.status == status, args
    lib.close()


# ------------------------------------------------------------------------------------------------
# NEXT-1: decode attention (n = 1, R = G rows per kv head), appended token by token
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("Hq,Hkv", [(4, 4), (8, 2)])
def test_decode_steps_append_one_token_at_a_time(Hq, Hkv):
    cfg = synth.GraftConfig("decode", 2, Hq, Hkv, 128, 16, 1e4, 3, 100, 300, 1000, 1, 3, 3, 0)
    wl, orc, lib, seg_ids = _pair(cfg, seed=1, tweak=_grow(8))
    task = wl.tasks[0]
    c_plans, o_plans = T.plans_of(wl, seg_ids)
    orc.stitch(o_plans)
    lib.stitch(c_plans)
    T0 = orc.tasks[0].n_tokens
    for step in range(4):
        out, ref = T.run_patch_both(orc, lib, cfg, task, 10 + step, positions=np.asarray([T0 + step], np.int32))
        T.assert_attn_close(out, ref, f"decode step {step}")
    _compare_task(orc, lib, 0, "after 4 decode steps")
    lib.close()


# ------------------------------------------------------------------------------------------------
# NEXT-3: two-tier residency -- offload to the pinned host tier, stitch from it in place, prefetch back
# ------------------------------------------------------------------------------------------------
def test_two_tier_residency_stitch_from_host_and_prefetch():
    B = _binding()
    cfg = synth.GraftConfig("tier", 2, 4, 2, 128, 16, 1e4, 5, 40, 160, 3000, 1, 4, 4, 0)
    wl = synth.make_workload(cfg, 1)
    total_pages = sum(-(-t.capacity // cfg.page_size) for t in wl.tasks)
    orc, lib, seg_ids = T.make_pair(cfg, wl, 1, n_pages=4 * total_pages, max_tasks=4, only_segments=list(range(5)),
                                    host_tier_tokens=int(wl.seg_lens.sum()))
    free0 = lib.pool_info()["segments_bytes_free"]
    used = [s for (s, _, _, _) in wl.tasks[0].entries]
    # offload two of the four segments of the plan: the stitch reads them over the host link, same result
    for s in used[:2]:
        lib.segment_offload(s), orc.segment_offload(s)
        lib.segment_offload(s)                                   # idempotent
        assert lib.segment_info(s) == orc.segment_info(s) == (int(wl.seg_lens[s]), int(wl.orig_starts[s]), False)
    assert lib.pool_info()["segments_bytes_free"] > free0
    c_plans, o_plans = T.plans_of(wl, seg_ids)
    orc.stitch(o_plans)
    lib.stitch(c_plans)
    T.compare_stitched(orc, lib, wl)
    # bring one back, release the other while offloaded; the arena accounting returns
    lib.segment_prefetch(used[0]), orc.segment_prefetch(used[0])
    assert lib.segment_info(used[0])[2] is True
    c_plans[0]["task_id"] = o_plans[0].task_id = 1
    orc.stitch(o_plans)
    lib.stitch(c_plans)
    wl.tasks[0].task_id = 1
    T.compare_stitched(orc, lib, wl)
    lib.segment_prefetch(used[1])
    assert lib.pool_info()["segments_bytes_free"] == free0
    lib.segment_offload(used[1])
    lib.segment_release(used[1]), orc.segment_release(used[1])
    k, v = synth.segment_kv(cfg, used[1], int(wl.seg_lens[used[1]]), 1, "cpu")
    assert lib.segment_register(k.cuda(), v.cuda(), 0) == orc.segment_register(synth.to_bits(k), synth.to_bits(v), 0) == used[1]
    # extraction from a cache stitched out of host-tier segments, then offload of the extracted segment
    spare = next(s for s in range(5) if s not in used)           # frees a table slot and an arena range
    lib.segment_release(spare), orc.segment_release(spare)
    sid = lib.segment_extract(1, 3, 20, 0)
    assert sid == orc.segment_extract(1, 3, 20, 0) == spare
    lib.segment_offload(sid), orc.segment_offload(sid)
    plan_c = {"task_id": 2, "entries": [(sid, 0, 20, 9)], "holes": [(0, 9)], "capacity_tokens": 29}
    orc.stitch([O.Plan(2, [O.PlanEntry(sid, 0, 20, 9)], [O.Hole(0, 9)], 29)])
    lib.stitch([plan_c])
    _compare_task(orc, lib, 2, "graft of an extracted, offloaded segment")
    st = lib.stats()
    assert st["offload_copies"] == 4 and st["prefetch_copies"] == 2
    with pytest.raises(B.FcgError) as e:
        lib.segment_offload(99)
    assert e.value.status == B.FCG_ERR_BAD_SEGMENT
    lib.close()
    # without a host tier the calls are refused
    orc, lib, seg_ids = T.make_pair(cfg, wl, 1, only_segments=[0])
    with pytest.raises(B.FcgError) as e:
        lib.segment_offload(0)
    assert e.value.status == B.FCG_ERR_INVALID_ARG
    lib.close()


# ------------------------------------------------------------------------------------------------
# NEXT-4: fcg_patch_rope -- q / k given before position encoding
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("rope_mode,D", [(1, 128), (2, 128), (1, 64), (0, 128), (1, 256), (2, 256), (1, 96), (2, 160), (1, 80)])
def test_patch_rope_matches_oracle(rope_mode, D):
    cfg = synth.GraftConfig("prope", 2, 8, 2, D, 16, 5e5, 3, 100, 300, 30000, 1, 3, 3, 0, holes=((0, 45), (-1, 50)))
    wl, orc, lib, seg_ids = _pair(cfg, seed=4, rope_mode=rope_mode)
    task = wl.tasks[0]
    c_plans, o_plans = T.plans_of(wl, seg_ids)
    orc.stitch(o_plans)
    lib.stitch(c_plans)
    # first the mid hole (45 consecutive positions: one exact anchor + a re-anchor after 32), then the end hole in two
    # calls with a gap pattern (non-consecutive positions are not allowed to leave holes: use consecutive chunks)
    holes = sorted(task.holes)
    chunks = [np.arange(holes[0][0], holes[0][0] + holes[0][1]), np.arange(holes[1][0], holes[1][0] + 7),
              np.arange(holes[1][0] + 7, holes[1][0] + holes[1][1])]
    for ci, pos in enumerate(chunks):
        pos = pos.astype(np.int32)
        q, k, v = synth.patch_qkv(cfg, 0, len(pos), 40 + ci, "cpu")
        ref = orc.patch_rope(0, 0, synth.to_bits(q), synth.to_bits(k), synth.to_bits(v), pos)
        out = lib.patch_rope(0, 0, q.cuda(), k.cuda(), v.cuda(), pos)
        torch.cuda.synchronize()
        T.assert_attn_close(out, ref, f"patch_rope chunk {ci}")
        ot = orc.tasks[0]
        for layer in range(cfg.n_layers):
            kg, vg = lib.task_read(0, layer, 0, ot.capacity)
            kb, vb = synth.to_bits(kg), synth.to_bits(vg)
            assert np.array_equal(vb[:, pos], ot.v[layer][:, pos]), "V scatter not bit-exact"
            if rope_mode == 0:
                assert np.array_equal(kb[:, pos], ot.k[layer][:, pos])
            else:
                T.assert_k_within_1ulp(kb[:, pos], ot.k[layer][:, pos], f"rotated patch K, chunk {ci} layer {layer}")
    assert lib.stats()["rope_qk_launches"] == (0 if rope_mode == 0 else len(chunks))
    B = _binding()
    with pytest.raises(B.FcgError) as e:
        lib.patch_rope(0, 0, q.cuda(), k.cuda(), v.cuda(), pos[::-1].copy())
    assert e.value.status == B.FCG_ERR_INVALID_ARG
    lib.close()


# ------------------------------------------------------------------------------------------------
# NEXT-4: boundary-recompute plan -- positions from the library, re-patched over the stitched cache
# ------------------------------------------------------------------------------------------------
def test_boundary_positions_and_repatch():
    cfg = synth.GraftConfig("bound", 2, 4, 2, 128, 16, 1e4, 5, 40, 120, 3000, 1, 4, 4, 0)
    wl, orc, lib, seg_ids = _pair(cfg, seed=6)
    task = wl.tasks[0]
    c_plans, o_plans = T.plans_of(wl, seg_ids)
    orc.stitch(o_plans)
    lib.stitch(c_plans)
    for width in (1, 4, 1000):
        assert lib.task_boundary_positions(0, width).tolist() == orc.task_boundary_positions(0, width)
    pos = lib.task_boundary_positions(0, 4)
    assert len(pos) == 4 * (len(task.entries) - 1)
    # the caller's recomputed tokens overwrite the stitched ones; every query sees its whole prefix
    out, ref = T.run_patch_both(orc, lib, cfg, task, 9, positions=pos)
    T.assert_attn_close(out, ref, "re-patch of the boundary tokens")
    T.compare_cache_bits(orc, lib, 0, pos)
    _compare_task(orc, lib, 0, "after the boundary re-patch")
    lib.close()
