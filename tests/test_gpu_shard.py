"""The sharded CUDA path on ONE GPU: the shards of a world of 2 are two
libraries in one process -- the same code `bench.py --shard head|task` runs with one library per rank -- compared with
the UNSHARDED oracle.  No collective is involved (the path needs none); the libraries never wait on one another.

* head-parallel: library r holds kv heads shard.kv_head_range(Hkv, r, 2) of every segment and of every cache, plans
  and page tables are replicated integers, outputs are concatenated along the head axis;
* task-parallel: library r grafts the tasks shard.assign_tasks gives it, over a replicated segment library.
"""
import numpy as np
import pytest
import torch

import fcg_testlib as T
from oracle import fcg_oracle as O
from paper_2606_13097_b200 import shard, synth

pytestmark = pytest.mark.gpu
WORLD = 2


def _cfg():
    return synth.GraftConfig("shard", 3, 8, 4, 128, 16, 1e4, 6, 80, 300, 2000, 5, 2, 4, 0, total_min=200, total_max=1200,
                             distinct_segments=False, holes=((0, 0), (-1, 0)), patch_min=3, patch_max=40)


def _oracle(cfg, wl, seed):
    orc = O.OracleLibrary(cfg.n_layers, cfg.n_q_heads, cfg.n_kv_heads, cfg.head_dim, page_size=cfg.page_size, rope_base=cfg.rope_base,
                          n_pages=4096)
    segs = {}
    for s in range(cfg.n_segments):
        k, v = synth.segment_kv(cfg, s, int(wl.seg_lens[s]), seed)
        segs[s] = (k, v)
        assert orc.segment_register(synth.to_bits(k), synth.to_bits(v), int(wl.orig_starts[s])) == s
    orc.stitch([O.Plan(t.task_id, [O.PlanEntry(*e) for e in t.entries], [O.Hole(*h) for h in t.holes], t.capacity) for t in wl.tasks])
    refs = {}
    for t in wl.tasks:
        q, k, v = synth.patch_qkv(cfg, t.task_id, len(t.positions), seed)
        refs[t.task_id] = (q, k, v, orc.patch(t.task_id, 0, synth.to_bits(q), synth.to_bits(k), synth.to_bits(v), t.positions))
    return orc, segs, refs


def _library(cfg_r, full_cfg, wl, tasks, segs, kv=None):
    from paper_2606_13097_b200.binding import FcgLibrary
    lib = FcgLibrary(n_layers=cfg_r.n_layers, n_q_heads=cfg_r.n_q_heads, n_kv_heads=cfg_r.n_kv_heads, head_dim=cfg_r.head_dim,
                     page_size=cfg_r.page_size, rope_base=cfg_r.rope_base, max_segments=full_cfg.n_segments,
                     max_tasks=max(t.task_id for t in wl.tasks) + 1, max_task_tokens=max(t.capacity for t in wl.tasks),
                     n_pages=sum(-(-t.capacity // cfg_r.page_size) for t in tasks) + 4, segment_tokens=int(wl.seg_lens.sum()))
    for s in range(full_cfg.n_segments):
        k, v = segs[s]
        if kv is not None:
            k, v = shard.slice_kv_heads(k, full_cfg.n_kv_heads, kv, WORLD, 1), shard.slice_kv_heads(v, full_cfg.n_kv_heads, kv, WORLD, 1)
        assert lib.segment_register(k.cuda(), v.cuda(), int(wl.orig_starts[s])) == s
    return lib


def test_head_parallel_shards_reproduce_the_unsharded_oracle():
    cfg, seed = _cfg(), 3
    wl = synth.make_workload(cfg, seed)
    orc, segs, refs = _oracle(cfg, wl, seed)
    G = cfg.n_q_heads // cfg.n_kv_heads
    libs = []
    for r in range(WORLD):
        cfg_r = shard.head_sharded_config(cfg, r, WORLD)
        assert cfg_r.n_kv_heads == cfg.n_kv_heads // WORLD and cfg_r.n_q_heads == cfg.n_q_heads // WORLD
        libs.append(_library(cfg_r, cfg, wl, wl.tasks, segs, kv=r))
    plans = [{"task_id": t.task_id, "entries": t.entries, "holes": t.holes, "capacity_tokens": t.capacity} for t in wl.tasks]
    ids = [t.task_id for t in wl.tasks]
    npt = [len(t.positions) for t in wl.tasks]
    pos = np.concatenate([t.positions for t in wl.tasks]).astype(np.int32)
    outs = []
    for r, lib in enumerate(libs):
        lib.stitch(plans)                                              # replicated integers: the same plans on every shard
        q = torch.cat([shard.slice_q_heads(refs[t][0], cfg.n_q_heads, cfg.n_kv_heads, r, WORLD) for t in ids], dim=1).cuda()
        k = torch.cat([shard.slice_kv_heads(refs[t][1], cfg.n_kv_heads, r, WORLD, 2) for t in ids], dim=1).cuda()
        v = torch.cat([shard.slice_kv_heads(refs[t][2], cfg.n_kv_heads, r, WORLD, 2) for t in ids], dim=1).cuda()
        outs.append(lib.patch_batch(ids, npt, 0, q.contiguous(), k.contiguous(), v.contiguous(), pos))
    torch.cuda.synchronize()
    whole = torch.cat(outs, dim=2)                                     # what shard.gather_head_outputs assembles over ranks
    ref = np.concatenate([refs[t][3] for t in ids], axis=1)
    T.assert_attn_close(whole, ref, "head-sharded outputs, concatenated")
    for r, lib in enumerate(libs):
        b, e = shard.kv_head_range(cfg.n_kv_heads, r, WORLD)
        for t in wl.tasks:
            ot = orc.tasks[t.task_id]
            assert np.array_equal(lib.task_page_table_host(t.task_id), np.asarray(ot.page_table, np.int32)), "page tables are replicated"
            for layer in range(cfg.n_layers):
                kg, vg = lib.task_read(t.task_id, layer, 0, t.capacity)
                f = ot.filled
                assert np.array_equal(synth.to_bits(vg)[:, f], ot.v[layer][b:e][:, f])
                T.assert_k_within_1ulp(synth.to_bits(kg)[:, f], ot.k[layer][b:e][:, f], f"shard {r} task {t.task_id} layer {layer}")
        lib.close()


def test_task_parallel_shards_reproduce_the_unsharded_oracle():
    cfg, seed = _cfg(), 4
    wl = synth.make_workload(cfg, seed)
    orc, segs, refs = _oracle(cfg, wl, seed)
    seen = []
    for r in range(WORLD):
        mine, assignment = shard.rank_workload(wl, r, WORLD, cfg.kv_bytes_per_token)
        tasks = [wl.tasks[i] for i in mine]
        seen += mine
        lib = _library(cfg, cfg, wl, tasks, segs)
        pages = O.PagePool(lib.pool_info()["n_pages"])          # what the rank's own pool hands out, tasks in plan order
        lib.stitch([{"task_id": t.task_id, "entries": t.entries, "holes": t.holes, "capacity_tokens": t.capacity} for t in tasks])
        ids = [t.task_id for t in tasks]
        npt = [len(t.positions) for t in tasks]
        pos = np.concatenate([t.positions for t in tasks]).astype(np.int32)
        q, k, v = [torch.cat([refs[t][j] for t in ids], dim=1).cuda().contiguous() for j in range(3)]
        out = lib.patch_batch(ids, npt, 0, q, k, v, pos)
        torch.cuda.synchronize()
        T.assert_attn_close(out, np.concatenate([refs[t][3] for t in ids], axis=1), f"rank {r}: tasks {ids}")
        for t in tasks:
            ot = orc.tasks[t.task_id]
            want = pages.allocate(-(-t.capacity // cfg.page_size))
            assert lib.task_page_table_host(t.task_id).tolist() == want
            for layer in (0, cfg.n_layers - 1):
                kg, vg = lib.task_read(t.task_id, layer, 0, t.capacity)
                f = ot.filled
                assert np.array_equal(synth.to_bits(vg)[:, f], ot.v[layer][:, f])
                T.assert_k_within_1ulp(synth.to_bits(kg)[:, f], ot.k[layer][:, f], f"rank {r} task {t.task_id}")
        lib.close()
    assert sorted(seen) == list(range(len(wl.tasks))), "every task belongs to exactly one rank"
