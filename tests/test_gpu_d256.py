"""head_dim 256 (R27; the paper's cross-family ablation includes Gemma, Table 4, whose heads are
256 wide): the cases the parametrised tests of the other files do not reach -- the lazy O-rescale branch of the
head_dim-256 kernel, many row groups of one task with KV splits, the attention policy (head_dim 256 has the tcgen05
kernel only), a length-changing patch and a segment extraction through stitch_kernel<256>."""
import numpy as np
import pytest
import torch

from oracle import fcg_oracle as O
from paper_2606_13097_b200 import synth
import fcg_testlib as T

pytestmark = pytest.mark.gpu
D = 256


def test_d256_growing_scores_force_the_rescale_path():
    """Scores that grow along the cache push the running row maximum up by more than the lazy-rescale threshold many
    times: the O-rescale branch (8 chunks of 32 TMEM columns at head_dim 256) must run, prefill-like and for short tails."""
    L, Hq, Hkv, T_ = 1, 4, 2, 700
    cfg = synth.GraftConfig("grow256", L, Hq, Hkv, D, 16, 1e4, 1, 8, 8, 0, 1, 1, 1, 0)
    wl = synth.make_workload(cfg, 1)
    wl.tasks[0].entries, wl.tasks[0].holes, wl.tasks[0].capacity = [], [(0, T_)], T_
    orc, lib, _ = T.make_pair(cfg, wl, 1, only_segments=[0], n_pages=T_ // 16 + 4)
    orc.stitch([O.Plan(0, [], [O.Hole(0, T_)], T_)])
    lib.stitch([{"task_id": 0, "entries": [], "holes": [(0, T_)], "capacity_tokens": T_}])
    g = torch.Generator().manual_seed(3)
    u = torch.rand(D, generator=g) + 0.5
    u = u / u.norm()
    ramp = torch.linspace(0.05, 1.0, T_)
    k = (u[None, None, None, :] * ramp[None, :, None, None] * 40.0).expand(L, T_, Hkv, D).to(torch.bfloat16).contiguous()
    q = (u[None, None, None, :] * 26.0).expand(L, T_, Hq, D).to(torch.bfloat16).contiguous()    # s up to 26*40/16 = 65
    v = torch.randn(L, T_, Hkv, D, generator=g).to(torch.bfloat16)
    pos = np.arange(T_, dtype=np.int32)
    ref = orc.patch(0, 0, synth.to_bits(q), synth.to_bits(k), synth.to_bits(v), pos)
    out = lib.patch(0, 0, q.cuda(), k.cuda(), v.cuda(), pos)
    torch.cuda.synchronize()
    assert lib.stats()["last_attn_path"] == 2
    T.assert_attn_close(out, ref, "head_dim 256 prefill-like, growing scores")
    for n in (1, 20, 100):
        sl = slice(T_ - n, T_)
        ref = orc.patch(0, 0, synth.to_bits(q[:, sl]), synth.to_bits(k[:, sl]), synth.to_bits(v[:, sl]), pos[sl])
        out = lib.patch(0, 0, q[:, sl].contiguous().cuda(), k[:, sl].contiguous().cuda(), v[:, sl].contiguous().cuda(), pos[sl])
        torch.cuda.synchronize()
        T.assert_attn_close(out, ref, f"head_dim 256 tail of {n} tokens, growing scores")
    lib.close()


@pytest.mark.parametrize("n,Hq,Hkv,ctx,P,splits", [(130, 2, 1, 2600, 16, 0), (260, 2, 2, 1500, 8, 2), (45, 8, 2, 1000, 64, 0),
                                                  (300, 2, 2, 777, 16, 3), (64, 16, 4, 4096, 32, 0), (1, 8, 1, 5000, 16, 5)])
def test_d256_row_groups_splits_and_forced_split_policy(n, Hq, Hkv, ctx, P, splits):
    """several 128-row groups per kv head, ragged last tiles, KV splits + combine<256>, a NaN-poisoned pool; asking for the
    split-KV mma.sync path (tc_min_rows = INT_MAX) still runs the tcgen05 kernel: head_dim 256 has no other."""
    L = 2
    cfg = synth.GraftConfig("rg256", L, Hq, Hkv, D, P, 5e5, 2, ctx, ctx, 1000, 1, 1, 1, 0, holes=((-1, n),))
    wl = synth.make_workload(cfg, n + ctx)
    orc, lib, seg_ids = T.make_pair(cfg, wl, 3, n_pages=-(-(ctx + 2 * n + 8) // P) + 4, max_task_tokens=ctx + 2 * n + 8, workspace_bytes=256 << 20)
    info = lib.pool_info()
    lib.arena[info["k_pool_offset"]: info["k_pool_offset"] + 2 * info["pool_bytes"]].view(torch.int16).fill_(0x7FC1)
    c_plans, o_plans = T.plans_of(wl, seg_ids)
    orc.stitch(o_plans)
    lib.stitch(c_plans)
    T.compare_stitched(orc, lib, wl)
    lib.set_attn_policy(2 ** 31 - 1, splits)
    task = wl.tasks[0]
    out, ref = T.run_patch_both(orc, lib, cfg, task, 5)
    st = lib.stats()
    assert st["last_attn_path"] == 2
    if splits:
        assert st["last_attn_splits"] == min(splits, -(-(ctx + n) // 64))
    assert torch.isfinite(out.float()).all()
    T.assert_attn_close(out, ref, "head_dim 256, patch at the end")
    T.compare_cache_bits(orc, lib, 0, task.positions)
    pos = np.arange(task.capacity, task.capacity + n, dtype=np.int32)          # appended: grows the task (R25)
    out, ref = T.run_patch_both(orc, lib, cfg, task, 6, positions=pos)
    T.assert_attn_close(out, ref, "head_dim 256, appended patch")
    lib.close()


@pytest.mark.parametrize("rope_mode", [1, 2])
def test_d256_shift_and_extract(rope_mode):
    """suffix re-graft (fcg_task_shift, both directions, one growing the task) and segment extraction through
    stitch_kernel<256>.  Every operation starts from cache rows written by the scatter (bit-exact on both sides), so each
    comparison is ONE rotation generation and the 1-ulp bar applies."""
    L, Hq, Hkv, P, T_ = 2, 4, 2, 16, 200
    cfg = synth.GraftConfig("shift256", L, Hq, Hkv, D, P, 1e4, 1, 60, 60, 0, 3, 1, 1, 0)
    wl = synth.make_workload(cfg, 11)
    for t in wl.tasks:
        t.entries, t.holes, t.capacity = [], [(0, T_)], T_
    orc, lib, _ = T.make_pair(cfg, wl, 11, rope_mode=rope_mode, n_pages=3 * 2 * (-(-(T_ + 64) // P)) + 8, max_task_tokens=T_ + 64, max_tasks=4,
                              only_segments=[0])
    lib.segment_release(0), orc.segment_release(0)              # the id and the arena range the extracted segment takes
    pos = np.arange(T_, dtype=np.int32)
    for t in wl.tasks:
        orc.stitch([O.Plan(t.task_id, [], [O.Hole(0, T_)], T_)])
        lib.stitch([{"task_id": t.task_id, "entries": [], "holes": [(0, T_)], "capacity_tokens": T_}])
        T.run_patch_both(orc, lib, cfg, t, 30 + t.task_id, positions=pos)
        T.compare_cache_bits(orc, lib, t.task_id, pos)

    def compare(task_id, what):
        ot = orc.tasks[task_id]
        assert np.array_equal(lib.task_page_table_host(task_id), np.asarray(ot.page_table, np.int32)), what
        for layer in range(L):
            k, v = lib.task_read(task_id, layer, 0, ot.capacity)
            f = ot.filled
            assert np.array_equal(synth.to_bits(v)[:, f], ot.v[layer][:, f]), f"{what}: V"
            T.assert_k_within_1ulp(synth.to_bits(k)[:, f], ot.k[layer][:, f], f"{what}, layer {layer}")

    mid = 97
    for task_id, (src, n, dst) in ((0, (mid, T_ - mid, mid + 21)), (1, (mid, T_ - mid, mid - 5))):
        orc.task_shift(task_id, src, n, dst)
        lib.task_shift(task_id, src, n, dst)
        torch.cuda.synchronize()
        compare(task_id, f"shift {src} -> {dst}")
    n_ext = 50
    sid_o = orc.segment_extract(2, 33, n_ext, 0)                # keys un-rotated by 33 positions: canonical form
    sid_g = lib.segment_extract(2, 33, n_ext, 0)
    assert sid_o == sid_g
    orc.stitch([O.Plan(3, [O.PlanEntry(sid_o, 0, n_ext, 0)], [], n_ext)])       # delta 0: a bit copy of the stored segment
    lib.stitch([{"task_id": 3, "entries": [(sid_g, 0, n_ext, 0)], "holes": [], "capacity_tokens": n_ext}])
    compare(3, "extracted segment")
    lib.close()
