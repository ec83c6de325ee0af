"""bench.py's host-side arithmetic (no GPU): algorithmic bytes / flops against hand values, the traffic table it reads
from profiles/, and the configuration tables."""
import numpy as np

import bench
from paper_2606_13097_b200 import synth


def test_algorithmic_bytes_and_flops_by_hand():
    cfg = synth.CONFIGS["C2"]
    wl = synth.make_workload(cfg, 1)
    assert wl.stitched_tokens == 4096 - 64 and wl.patch_tokens == 64
    # C2: 32 layers x 32 kv heads x 128 x 2 B x (K, V) = 512 KiB per token; stitched bytes are read once and written once
    assert cfg.kv_bytes_per_token == 512 * 1024
    assert bench.stitch_bytes(cfg, wl) == 4032 * 1024 * 1024
    # the last patch position is 4095: 4096 visible tokens x 512 KiB, read once
    assert bench.attn_bytes(cfg, wl) == 4096 * 512 * 1024
    # flops: per layer, q head and patch token 4 D (p + 1); positions = 16 in the mid hole + 48 at the end
    pos = np.asarray(wl.tasks[0].positions, np.int64)
    assert bench.attn_flops(cfg, wl) == 4 * 128 * 32 * 32 * int((pos + 1).sum())
    assert bench.attn_rows(cfg, wl) == 64
    # a subset of tasks (sharded runs) counts only those tasks
    c4 = synth.CONFIGS["C4"]
    w4 = synth.make_workload(c4, 1)
    assert bench.stitch_bytes(c4, w4, w4.tasks[:3]) + bench.stitch_bytes(c4, w4, w4.tasks[3:]) == bench.stitch_bytes(c4, w4)
    assert bench.attn_rows(c4, w4) == max(len(t.positions) for t in w4.tasks) * 4


def test_traffic_table_is_read_from_profiles():
    traffic, src = bench.ncu_traffic()
    assert src is not None and src.startswith("profiles/") and src.endswith("_traffic.csv")
    for name in ("C2", "C3", "C4", "C5"):
        assert traffic[name]["stitch"] > 1e9 and traffic[name]["attn"] > 1e9
    # ncu's DRAM bytes of the stitch agree with the algorithmic bytes within a few per cent (no re-reads)
    cfg = synth.CONFIGS["C2"]
    assert abs(traffic["C2"]["stitch"] / bench.stitch_bytes(cfg, synth.make_workload(cfg, 1)) - 1) < 0.05


def test_bench_configs():
    assert set(bench.ALL_CONFIGS) <= set(synth.CONFIGS) and bench.HEADLINE in bench.ALL_CONFIGS
    d = bench.BENCH_CONFIGS["D64"]
    assert d.head_dim == 64 and d.total_tokens == 4096
    wl = synth.make_workload(d, 1)
    assert wl.tasks[0].capacity == 4096 and len(wl.tasks[0].positions) == 16
