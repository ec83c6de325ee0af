"""Round-3 GPU tests: regressions found by review of the host-side planner (ordering of the scratch area, patch plans)."""
import numpy as np
import pytest
import torch

from paper_2606_13097_b200 import synth
import fcg_testlib as T

pytestmark = pytest.mark.gpu


def test_host_patch_right_after_a_split_patch_with_large_partials():
    """fcg_patch_host stages q / k / v at the END of the scratch area from the library's copy stream, which is not ordered
    after `stream`.  A preceding split-KV fcg_patch whose fp32 partials reach into that area (small workspace, many
    splits) must have been read by its combine kernel before the copies land.  The stream is kept busy first, so the copy
    stream WOULD run ahead of the partial writes if nothing ordered it; both calls are then checked against the oracle."""
    L, Hq, Hkv, D, P = 6, 8, 2, 128, 16
    cfg = synth.GraftConfig("staging", L, Hq, Hkv, D, P, 5e5, 2, 1000, 1200, 4000, 1, 2, 2, 0, holes=((0, 64), (-1, 128)))
    wl = synth.make_workload(cfg, 5)
    orc, lib, seg_ids = T.make_pair(cfg, wl, 5, workspace_bytes=32 << 20)         # scratch = 16 MiB after the plan blobs
    c_plans, o_plans = T.plans_of(wl, seg_ids)
    orc.stitch(o_plans)
    lib.stitch(c_plans)
    task = wl.tasks[0]
    (mb, mn), (eb, en) = task.holes
    assert (mn, en) == (64, 128)
    mid, end = np.arange(mb, mb + mn, dtype=np.int32), np.arange(eb, eb + en, dtype=np.int32)
    q1, k1, v1 = synth.patch_qkv(cfg, 0, mn, 21, "cpu")
    q2, k2, v2 = synth.patch_qkv(cfg, 0, en, 22, "cpu")
    ref1 = orc.patch(0, 0, synth.to_bits(q1), synth.to_bits(k1), synth.to_bits(v1), mid)
    ref2 = orc.patch(0, 0, synth.to_bits(q2), synth.to_bits(k2), synth.to_bits(v2), end)
    d1 = [x.cuda().contiguous() for x in (q1, k1, v1)]
    h2 = [x.contiguous().pin_memory() for x in (q2, k2, v2)]
    out2 = torch.empty_like(h2[0]).pin_memory()
    out2.fill_(float("nan"))
    # warm-up: the same two calls once, unhurried (the first launch of a kernel loads it, which blocks the host until the
    # device is idle and would let the busy stream below drain before anything else is enqueued)
    lib.set_attn_policy(1, 14)
    lib.patch(0, 0, *d1, mid)
    lib.set_attn_policy(1, 1)
    lib.patch_host(0, 0, *h2, end, out2)
    torch.cuda.synchronize()
    out2.fill_(float("nan"))
    lib.set_attn_policy(1, 14)            # asks for 14 splits; whole 64-token tiles per split make it 9 for this cache length
    torch.cuda._sleep(300_000_000)        # ~0.15 s: everything below is enqueued while the stream is still busy
    out1 = lib.patch(0, 0, *d1, mid)
    ns = lib.stats()["last_attn_splits"]
    scratch = (32 << 20) - (16 << 20)     # workspace minus the 16 plan-blob slots of 1 MiB
    partials = L * ns * mn * Hq * (D + 2) * 4                                    # 6 x 9 x 64 x 8 rows x 130 fp32 = 14.4 MB
    staging = 2 * (L * en * Hq * D * 2) + 2 * (L * en * Hkv * D * 2)             # q, out, k, v of the host call: 3.75 MiB
    assert ns > 1 and scratch - staging < partials <= scratch, (ns, partials, staging)   # the two regions do overlap
    lib.set_attn_policy(1, 1)             # the host call itself runs with one split (no partials of its own)
    lib.patch_host(0, 0, *h2, end, out2)
    torch.cuda.synchronize()
    T.assert_attn_close(out1, ref1, "split patch before the host call")
    T.assert_attn_close(out2, ref2, "host call right after the split patch")
    lib.close()


def test_plans_are_invalidated_by_task_shift_and_freed_with_the_library():
    """A plan compares task generations only; fcg_task_shift un-fills source positions and re-pages the destination, so
    it must bump the generation (a planned call would otherwise attend over positions that are no longer filled, R6).
    Plans the caller leaves behind go with the library; destroying one twice is refused."""
    from paper_2606_13097_b200 import binding as B
    L, Hq, Hkv, D, P = 2, 4, 2, 128, 16
    cfg = synth.GraftConfig("planshift", L, Hq, Hkv, D, P, 1e4, 2, 200, 300, 2000, 1, 2, 2, 0, holes=((-1, 24),))
    wl = synth.make_workload(cfg, 3)
    orc, lib, seg_ids = T.make_pair(cfg, wl, 3, n_pages=128, max_task_tokens=1024)
    c_plans, _ = T.plans_of(wl, seg_ids)
    lib.stitch(c_plans)
    task = wl.tasks[0]
    n = len(task.positions)
    q, k, v = [x.cuda() for x in synth.patch_qkv(cfg, 0, n, 1)]
    out = torch.empty_like(q)
    plan = lib.patch_plan_create([0], [n], task.positions, 1)
    lib.patch_planned(plan, 0, q[:1], k[:1], v[:1], out[:1])
    lib.patch_plan_create([0], [n], task.positions, 1)                      # a second plan, never destroyed by the caller
    first_len = task.entries[0][2]
    lib.task_shift(0, first_len // 2, 8, int(task.positions[-1]) + 40)      # move 8 stitched tokens past the end
    with pytest.raises(B.FcgError) as e:
        lib.patch_planned(plan, 1, q[1:], k[1:], v[1:], out[1:])
    assert e.value.status == B.FCG_ERR_BAD_TASK
    lib.patch_plan_destroy(plan)
    with pytest.raises(B.FcgError) as e:
        lib.patch_plan_destroy(plan)
    assert e.value.status == B.FCG_ERR_INVALID_ARG
    # the second plan is still live when the library goes away: it is freed with it (no crash; the arena is the caller's)
    torch.cuda.synchronize()
    lib.close()


def test_failing_calls_enqueue_nothing():
    """fcg.h: every host-side check of a call happens before any copy or launch.  (a) a stitch whose plan blob would exceed
    1 MiB (12 000 one-token entries) is refused with the library unchanged and usable; (b) a host patch whose split
    partials do not fit beside its staging area is refused before its host->device copies: nothing was counted as launched,
    the output buffer is untouched and the same call succeeds with fewer splits."""
    from paper_2606_13097_b200 import binding as B
    # (a)
    lib = B.FcgLibrary(n_layers=1, n_q_heads=1, n_kv_heads=1, head_dim=16, max_segments=2, max_tasks=2, max_task_tokens=12032,
                       n_pages=800, segment_tokens=64)
    k = torch.randn(1, 1, 16, 16).to(torch.bfloat16).cuda()
    seg = lib.segment_register(k, k.clone(), 0)
    big = {"task_id": 0, "entries": [(seg, i % 16, 1, i) for i in range(12000)], "holes": [], "capacity_tokens": 12000}
    before = (lib.pool_info(), lib.stats())
    with pytest.raises(B.FcgError) as e:
        lib.stitch([big])
    assert e.value.status == B.FCG_ERR_OUT_OF_ARENA and "plan blob" in str(e.value)
    assert (lib.pool_info(), lib.stats()) == before
    lib.stitch([{"task_id": 0, "entries": [(seg, 0, 16, 0)], "holes": [], "capacity_tokens": 16}])
    kk, _ = lib.task_read(0, 0, 0, 16)
    assert torch.equal(kk.view(torch.int16), k[0].view(torch.int16))
    lib.close()
    # (b)
    L, Hq, Hkv, D, P = 6, 8, 2, 128, 16
    cfg = synth.GraftConfig("dry", L, Hq, Hkv, D, P, 5e5, 2, 1000, 1200, 4000, 1, 2, 2, 0, holes=((-1, 128),))
    wl = synth.make_workload(cfg, 5)
    orc, lib, seg_ids = T.make_pair(cfg, wl, 5, workspace_bytes=32 << 20)
    c_plans, o_plans = T.plans_of(wl, seg_ids)
    orc.stitch(o_plans)
    lib.stitch(c_plans)
    pos = wl.tasks[0].positions
    q, k, v = synth.patch_qkv(cfg, 0, len(pos), 3, "cpu")
    ref = orc.patch(0, 0, synth.to_bits(q), synth.to_bits(k), synth.to_bits(v), pos)
    h = [x.contiguous().pin_memory() for x in (q, k, v)]
    out = torch.empty_like(h[0]).pin_memory()
    out.fill_(float("nan"))
    lib.set_attn_policy(1, 12)            # 128 tokens x 12 splits x 6 layers x 8 heads x 130 fp32 = 38 MB of partials: no room
    before = lib.stats()
    with pytest.raises(B.FcgError) as e:
        lib.patch_host(0, 0, *h, pos, out)
    assert e.value.status == B.FCG_ERR_OUT_OF_ARENA
    torch.cuda.synchronize()
    assert lib.stats() == before and bool(torch.isnan(out.float()).all())
    with pytest.raises(B.FcgError) as e:  # the rope variant checks before it launches its rotation kernel
        lib.patch_rope(0, 0, *[x.cuda() for x in (q, k, v)], pos)
    assert e.value.status == B.FCG_ERR_OUT_OF_ARENA and lib.stats() == before
    lib.set_attn_policy(1, 1)
    lib.patch_host(0, 0, *h, pos, out)
    torch.cuda.synchronize()
    T.assert_attn_close(out, ref, "host patch after the refused one")
    lib.close()


def test_bench_two_ranks_on_one_gpu_prints_a_compact_last_line():
    """Readiness for the day the scaling run happens: `bench.py --gpus 2` spawns two ranks (here both on cuda:0 with gloo as
    the control plane, so the ranks' kernels never wait on one another), shards the workload and has rank 0 print the compact
    headline as the LAST stdout line, the fat record before it on a DETAIL line."""
    import json
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    r = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--devices", "same", "--config", "C2", "--steps", "2",
                        "--no-seeds", "--no-next", "--no-cpu-baseline"], capture_output=True, text=True, timeout=540, cwd=root)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.strip()]
    last = lines[-1]
    assert len(last) < 4096 and any(ln.startswith("DETAIL ") for ln in lines[:-1])
    rec = json.loads(last)
    assert rec["n_gpus"] == 2 and rec["steps"] == 2 and rec["value"] > 0 and rec["scaling"] in ("weak", "strong")
    assert rec["gpu_launches"] > 0 and rec["roofline"]["frac"] > 0 and rec["e2e"]["h2d_bytes_per_step"] > 0
