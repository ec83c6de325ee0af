"""Fuzz campaign for patch attention (a campaign driver; tests/test_gpu_fuzz.py runs a bounded, fixed-seed slice of it): random geometry, patch placement, KV-split count and
kernel policy against the oracle -- the ragged edges of the CTA classes (rows per kv head around 32 / 64 / 128 / 256, a last
KV tile or split of a few tokens, holes in the middle of the cache, appends that grow the task), NaN-poisoned pool.

    python tests/fuzz_attention.py <campaign seed> <number of cases>        (needs a GPU)
"""
import os
import sys
import traceback

import numpy as np
import torch

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(HERE))
sys.path.insert(0, HERE)
import fcg_testlib as T  # noqa: E402
from paper_2606_13097_b200 import synth  # noqa: E402


def one_case(rng):
    D = int(rng.choice([64, 128, 256, 16, 32, 48, 80, 96, 112, 144, 160, 176, 192, 208, 224, 240]))
    Hkv = int(rng.choice([1, 2, 4]))
    G = int(rng.choice([1, 2, 4, 8]))
    Hq = Hkv * G
    P = int(rng.choice([8, 16, 32, 64]))
    L = int(rng.integers(1, 3))
    target_rows = int(rng.choice([1, 2, 7, 31, 32, 33, 63, 64, 65, 127, 128, 129, 200, 255, 256, 257, 300, 513]))
    n = max(1, -(-target_rows // G) if rng.random() < 0.5 else target_rows // G)
    ctx = int(rng.choice([1, 17, 63, 64, 65, 127, 128, 129, 500, 1000, 1999, 2600]))
    n_mid = int(rng.integers(0, n)) if (rng.random() < 0.4 and ctx > 3) else 0        # part of the patch in a hole mid-cache
    splits = int(rng.choice([0, 0, 0, 1, 2, 3, 5]))
    tc_min_rows = 1 if (D == 256 or rng.random() < 0.8) else 2 ** 31 - 1
    params = dict(D=D, Hq=Hq, Hkv=Hkv, P=P, L=L, n=n, ctx=ctx, n_mid=n_mid, splits=splits, tc_min_rows=tc_min_rows)
    holes = ((-1, n - n_mid),) if n_mid == 0 else ((0, n_mid), (-1, n - n_mid))
    n_seg = 2 if ctx >= 2 else 1
    per = -(-ctx // n_seg) + ctx // 6 + 2          # room for the sub-range starts synth skips (up to 1/8 of a segment)
    cfg = synth.GraftConfig("fuzz", L, Hq, Hkv, D, P, 1e4, n_seg, per, per, 3000, 1, n_seg, n_seg, ctx + n, holes=holes)
    wl = synth.make_workload(cfg, int(rng.integers(1, 10 ** 6)))
    task = wl.tasks[0]
    cap = task.capacity
    orc, lib, seg_ids = T.make_pair(cfg, wl, 3, n_pages=-(-(cap + n + 8) // P) + 4, max_task_tokens=cap + n + 8, workspace_bytes=256 << 20)
    try:
        info = lib.pool_info()
        lib.arena[info["k_pool_offset"]: info["k_pool_offset"] + 2 * info["pool_bytes"]].view(torch.int16).fill_(0x7FC1)
        c_plans, o_plans = T.plans_of(wl, seg_ids)
        orc.stitch(o_plans)
        lib.stitch(c_plans)
        lib.set_attn_policy(tc_min_rows, splits)
        out, ref = T.run_patch_both(orc, lib, cfg, task, 5)
        assert torch.isfinite(out.float()).all(), "non-finite output"
        T.assert_attn_close(out, ref, f"patch {params}")
        T.compare_cache_bits(orc, lib, 0, task.positions)
        pos = np.arange(cap, cap + n, dtype=np.int32)                     # appended: grows the task
        out, ref = T.run_patch_both(orc, lib, cfg, task, 6, positions=pos)
        T.assert_attn_close(out, ref, f"appended patch {params}")
    finally:
        lib.close()
    return params


def main(campaign_seed: int, n_cases: int) -> int:
    rng = np.random.default_rng(campaign_seed)
    fails = 0
    for i in range(n_cases):
        state = rng.bit_generator.state
        try:
            one_case(rng)
        except Exception as e:
            fails += 1
            print("FAIL case", i, repr(e)[:400], flush=True)
            traceback.print_exc()
            rng.bit_generator.state = state
            rng.integers(1 << 30)          # move on from the failing draw
    print(f"done: {n_cases} cases, {fails} failures")
    return fails


if __name__ == "__main__":
    sys.exit(1 if main(int(sys.argv[1]), int(sys.argv[2])) else 0)
