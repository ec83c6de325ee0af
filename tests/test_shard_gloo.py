"""N > 1 host logic on CPU: world_size-2 `gloo` processes shard a small grafting workload by task and by kv
head (paper_2606_13097_b200/shard.py), run each shard through the ORACLE (there is no GPU here, and the CUDA
path has no CPU fallback), exchange only the results, and must reproduce the unsharded oracle output bit for
bit.  This pins the sharding claims of DESIGN.md "Multi-GPU": tasks and kv heads are independent, so no
data-path collective is needed."""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

from paper_2606_13097_b200 import shard, synth  # noqa: E402

CFG = synth.scaled(synth.C4, name="C4-mini", n_layers=2, n_q_heads=8, n_kv_heads=4, head_dim=64, n_segments=6,
                   seg_len_min=24, seg_len_max=80, n_tasks=5, n_entries_min=2, n_entries_max=4, total_min=60, total_max=400,
                   patch_min=3, patch_max=9, orig_start_max=500)
SEED = 2


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _oracle_run(cfg, wl, task_idx, seg_slice, qkv_slice):
    """Oracle stitch + patch of the tasks `task_idx` on a (possibly head-sliced) library.  Returns float64 outputs
    concatenated over those tasks, the stitched K/V bits per task and the page tables."""
    from oracle import fcg_oracle as O
    orc = O.OracleLibrary(cfg.n_layers, cfg.n_q_heads, cfg.n_kv_heads, cfg.head_dim, page_size=cfg.page_size, rope_base=cfg.rope_base)
    for s in range(len(wl.seg_lens)):
        k, v = seg_slice(s)
        assert orc.segment_register(synth.to_bits(k), synth.to_bits(v), int(wl.orig_starts[s])) == s
    tasks = [wl.tasks[i] for i in task_idx]
    orc.stitch([O.Plan(t.task_id, [O.PlanEntry(*e) for e in t.entries], [O.Hole(*h) for h in t.holes], t.capacity) for t in tasks])
    outs, caches = [], {}
    for t in tasks:
        q, k, v = qkv_slice(t)
        outs.append(orc.patch(t.task_id, 0, synth.to_bits(q), synth.to_bits(k), synth.to_bits(v), t.positions))
        caches[t.task_id] = (orc.tasks[t.task_id].k.copy(), orc.tasks[t.task_id].v.copy())
    return (np.concatenate(outs, axis=1) if outs else np.zeros((cfg.n_layers, 0, cfg.n_q_heads, cfg.head_dim))), caches


def _full_inputs(wl):
    full = synth.scaled(CFG)
    segs = [synth.segment_kv(full, s, int(wl.seg_lens[s]), SEED) for s in range(full.n_segments)]
    qkv = {t.task_id: synth.patch_qkv(full, t.task_id, len(t.positions), SEED) for t in wl.tasks}
    return segs, qkv


def _worker(rank: int, world: int, port: int, q):
    try:
        sys.path.insert(0, ROOT)
        os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
        dist.init_process_group("gloo", rank=rank, world_size=world)
        wl = synth.make_workload(CFG, SEED)
        segs, qkv = _full_inputs(wl)
        n_per_task = [len(t.positions) for t in wl.tasks]

        # ---- task-parallel: every rank grafts its own tasks against the whole (replicated) library ----
        mine, assignment = shard.rank_workload(wl, rank, world, CFG.kv_bytes_per_token)
        out_t, _ = _oracle_run(CFG, wl, mine, lambda s: segs[s], lambda t: qkv[t.task_id])
        full_t = shard.gather_task_outputs(torch.from_numpy(out_t), mine, n_per_task, assignment)

        # ---- head-parallel: every rank grafts all tasks on its kv heads ---------------------------------
        sub = shard.head_sharded_config(CFG, rank, world)
        out_h, caches_h = _oracle_run(
            sub, wl, list(range(len(wl.tasks))),
            lambda s: tuple(shard.slice_kv_heads(x, CFG.n_kv_heads, rank, world, 1) for x in segs[s]),
            lambda t: (shard.slice_q_heads(qkv[t.task_id][0], CFG.n_q_heads, CFG.n_kv_heads, rank, world),
                       shard.slice_kv_heads(qkv[t.task_id][1], CFG.n_kv_heads, rank, world, 2),
                       shard.slice_kv_heads(qkv[t.task_id][2], CFG.n_kv_heads, rank, world, 2)))
        full_h = shard.gather_head_outputs(torch.from_numpy(out_h))
        t_max = shard.max_over_ranks(1.0 + rank)
        if rank == 0:
            q.put(("ok", full_t.numpy(), full_h.numpy(), t_max, assignment,
                   {tid: (k[:, :1].copy(), v[:, :1].copy()) for tid, (k, v) in caches_h.items()}))
        dist.barrier()
        dist.destroy_process_group()
    except Exception as e:  # pragma: no cover - reported to the parent
        import traceback
        q.put(("err", f"rank {rank}: {e}\n{traceback.format_exc()}"))


def test_task_and_head_sharding_reproduce_the_unsharded_oracle_over_gloo():
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = q.get(timeout=240)
    for p in procs:
        p.join(timeout=60)
    assert res[0] == "ok", res[1]
    _, full_t, full_h, t_max, assignment, caches0 = res

    wl = synth.make_workload(CFG, SEED)
    segs, qkv = _full_inputs(wl)
    ref, caches = _oracle_run(CFG, wl, list(range(len(wl.tasks))), lambda s: segs[s], lambda t: qkv[t.task_id])
    assert full_t.shape == ref.shape and np.array_equal(full_t, ref), "task-parallel shards do not reproduce the whole"
    assert full_h.shape == ref.shape and np.array_equal(full_h, ref), "head-parallel shards do not reproduce the whole"
    # rank 0's head shard of the stitched + patched cache is the matching slice of the whole cache
    for tid, (k0, v0) in caches0.items():
        assert np.array_equal(k0, caches[tid][0][:, :1]) and np.array_equal(v0, caches[tid][1][:, :1])
    assert t_max == 2.0
    assert sorted(i for a in assignment for i in a) == list(range(len(wl.tasks)))


def test_assign_tasks_is_balanced_and_deterministic():
    rng = np.random.default_rng(0)
    costs = rng.integers(1, 1000, size=37).tolist()
    for world in (1, 2, 3, 8):
        a = shard.assign_tasks(costs, world)
        assert a == shard.assign_tasks(costs, world)
        assert sorted(i for m in a for i in m) == list(range(37))
        loads = [sum(costs[i] for i in m) for m in a]
        assert max(loads) - min(loads) <= max(costs)          # LPT bound
    assert shard.assign_tasks([5, 5, 5], 2) == [[0, 2], [1]]
    with pytest.raises(ValueError):
        shard.assign_tasks([1], 0)


def test_head_ranges_partition_the_heads():
    for hkv, hq, world in [(8, 32, 1), (8, 32, 2), (8, 64, 8), (32, 32, 4)]:
        kv = [shard.kv_head_range(hkv, r, world) for r in range(world)]
        qh = [shard.q_head_range(hq, hkv, r, world) for r in range(world)]
        assert kv[0][0] == 0 and kv[-1][1] == hkv and all(kv[i][1] == kv[i + 1][0] for i in range(world - 1))
        assert qh[0][0] == 0 and qh[-1][1] == hq and all(qh[i][1] == qh[i + 1][0] for i in range(world - 1))
        g = hq // hkv
        for (kb, ke), (qb, qe) in zip(kv, qh):       # q head h maps to kv head h // G inside the same shard
            assert all(kb <= h // g < ke for h in range(qb, qe))
    with pytest.raises(ValueError):
        shard.kv_head_range(8, 0, 3)
    sub = shard.head_sharded_config(synth.C3, 1, 4)
    assert (sub.n_kv_heads, sub.n_q_heads, sub.n_layers) == (2, 8, synth.C3.n_layers)
    ts = shard.token_slices([3, 0, 5])
    assert [(s.start, s.stop) for s in ts] == [(0, 3), (3, 3), (3, 8)]
