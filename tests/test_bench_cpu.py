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


def _canned_record():
    """the shape of run_cuda's full record (long strings, six configurations with seeds and NEXT rows, a NaN)"""
    roof = {"kernel": "stitch_kernel (fused gather + RoPE-shift)", "bound": "hbm", "achieved": 6524.123456789, "peak": 6540.8,
            "unit": "GB/s", "frac": 0.99745, "peak_source": "measured (MEASURED_PEAKS.json, torch copy_ read+write)",
            "frac_of_8TBps": 0.8155, "traffic": 30110000000.0,
            "patch_attention": {"kernel": "attn_tc_kernel (tcgen05 / TMEM)", "bound": "hbm", "achieved": 4922.3333333, "peak": 6540.8,
                                "unit": "GB/s", "frac": 0.7526, "frac_of_8TBps": 0.6153, "rows_per_kv_head": 1024,
                                "flop_per_byte": 123.456, "TFLOPs": 601.2, "traffic": 15900000000.0,
                                "note": "timed as scatter + attention (+ combine); scatter is ~1 % of it"}}
    clocks = {"sm_mhz": 1882.0, "sm_min_mhz": 1777.0, "sm_max_mhz": 1965.0, "power_w_max": 573.836, "reasons": ["sw_power_cap"],
              "samples": 53, "window": "timed region", "source": "NVML polled every 4 ms " * 5}
    e2e = {"value": 4299.123, "unit": bench.UNIT, "ms_per_step": 10.84, "h2d_bytes_per_step": 367001600, "d2h_bytes_per_step": 245366784}
    per = {"workload": "x" * 300, "ms_per_step": 7.929, "steps": 20, "value_GBps": 5879.1, "stitch_ms": 4.751, "patch_ms": 3.17,
           "roofline": roof, "clocks": clocks, "e2e": e2e, "l2": "inputs larger than L2 (each step streams >= 1 GiB; no flush needed)",
           "seeds": {str(s): {"ms_per_step": 7.9, "stitch_ms": 4.7, "patch_ms": 3.2, "stitch_frac": 0.99, "patch_frac": 0.75} for s in (1, 2, 3)},
           "next_rows": {f"row{i}": {"ms": 0.1234567 * i, "GBps": 5632.0264, "bytes": 704643072, "note": "n" * 120} for i in range(12)}}
    res = {"metric": bench.METRIC, "value": 5879.123456, "unit": bench.UNIT, "n_gpus": 1, "steps": 20, "warmup": 5, "ms_per_step": 7.929,
           "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
           "config": {"workload": bench.short_workload("C4", synth.CONFIGS["C4"], 32, 118231, 2201, 1), "workload_long": "y" * 400,
                      "l2": per["l2"], "stitch_ms": 4.751, "stitch_ms_min": 4.7, "stitch_ms_median": 4.75, "patch_ms": 3.17,
                      "patch_ms_min": 3.1, "patch_ms_median": 3.16, "stitch_bytes": 30994000000, "attn_bytes": 15620000000,
                      "attn_flops": 1234567890123456, "attn_path": 2, "attn_splits": 1, "parallelism": "1 GPU", "traffic_source": "profiles/r02_traffic.csv"},
           "gpu_launches": 100, "roofline": roof, "clocks": clocks, "e2e": e2e,
           "cpu_baseline": {"value": 0.2475, "unit": bench.UNIT, "cores": 16, "host_cpus": 224, "kind": "oracle", "seconds": float("nan"),
                            "sample": "task 0 of C4, 1 of 32 layer(s) x 2 of 8 kv heads: " + "z" * 300},
           "prefill_compare": {"tokens": 32768, "graft_ms": 13.2, "own_kernel_ms_all_layers": 710.0, "torch_sdpa_ms_all_layers": 565.0,
                               "own_kernel_TFLOPs": 1234.5, "flops_all_layers": 10 ** 15, "torch_sdpa_note": "library kernel, context only"},
           "next_rows": per["next_rows"],
           "configs": {n: dict(per) for n in ("C4", "C2", "C3", "C5", "D64", "D256")}}
    res["configs"]["C1"] = {"error": "RuntimeError('" + "e" * 200 + "')"}
    return res


def test_headline_line_is_compact_strict_json():
    import json
    res = _canned_record()
    assert len(json.dumps(bench._sig(res, 7))) > 20000            # the fat record really is fat
    h = bench.headline(res)
    line = json.dumps(h, allow_nan=False)                         # strict JSON: NaN / Infinity would raise here
    assert len(line) < bench.HEADLINE_MAX_BYTES, len(line)
    back = json.loads(line)
    for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
                "dtype", "data", "gpu_launches", "config", "roofline", "cpu_baseline", "clocks", "e2e", "prefill_compare", "configs_summary"):
        assert key in back, key
    assert back["value"] > 0 and len(back["config"]["workload"]) <= 120
    assert set(back["roofline"]) >= {"bound", "achieved", "peak", "unit", "frac", "traffic", "patch_attention"}
    assert set(back["e2e"]) >= {"value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step"}
    assert set(back["cpu_baseline"]) >= {"value", "unit", "cores", "kind", "sample"} and back["cpu_baseline"]["seconds"] is None
    assert abs(back["prefill_compare"]["ratio"] - 710.0 / 13.2) < 0.01
    assert len(back["configs_summary"]) == 7 and len(back["configs_summary"]["C2"]) == 6
    assert "configs" not in back and "next_rows" not in back
    # a record that would still be too long loses its optional parts instead of overflowing
    res["configs"] = {f"X{i}": dict(res["configs"]["C4"]) for i in range(60)}
    assert len(json.dumps(bench.headline(res), allow_nan=False)) < bench.HEADLINE_MAX_BYTES
