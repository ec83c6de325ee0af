"""bench.py -- one "step" = one pass of the whole grafting hot path (S2 plan -> S3 fused gather +
RoPE-shift -> S4 scatter -> S5/S6 patch attention, all layers) over one synthetic batch.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config all|C1..C5] [--impl reference] [--shard ...]

Prints ONE JSON line (rank 0).  metric = BASELINE.json's: graft latency (ms_per_step) and achieved algorithmic HBM
GB/s (value) against the roofline on a B200.  With the default `--config all` the headline (value, ms_per_step,
roofline, e2e, config.workload) is C4 -- BASELINE.json configs[3], the largest configuration that exercises both
north_star kernels -- timed for EXACTLY K steps, and the key `configs` carries C2, C3, C4, C5 (and C1 as latency only)
with per-config stitch / patch times, algorithmic bytes and flops, roofline fractions, ncu traffic (read from
profiles/*.csv), end-to-end time, clock samples of that config's own timed region and layout seeds 1, 2, 3; C5 also
carries the graft-vs-prefill comparison BASELINE.json asks for.

Multi-GPU (`--gpus N` spawns N ranks through torch.distributed.run unless it already runs under it): the path shards
by task and by kv head with no data-path collective (paper_2606_13097_b200/shard.py).  Default at N > 1: the batched
configuration with 32 x N tasks, balanced over the ranks longest-first ("scaling": "weak"); `--shard task|head` split
the fixed single-GPU workload instead ("strong"); `--shard replica` runs N identical copies.
--impl reference times the CPU oracle (the only reference this paper has) on a bounded sample of the headline workload.
"""
from __future__ import annotations

import argparse
import csv
import json
import math
import os
import subprocess
import sys
import threading
import time

import numpy as np
import torch

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2606_13097_b200 import shard, synth  # noqa: E402

METRIC = "graft latency ms + HBM GB/s (stitch+RoPE shift, patch attn) vs roofline, 1 B200"
UNIT = "GB/s (algorithmic, whole graft)"
FALLBACK_HBM_GBS = 6650.0          # B200_PROFILING.md fallback, used only if MEASURED_PEAKS.json is absent
FALLBACK_BF16_SUSTAINED = 1400.0
HEADLINE = "C4"
ALL_CONFIGS = ("C4", "C2", "C3", "C5")
EXTRACT_TOKENS = 1024
# not a BASELINE.json configuration: the head_dim-64 geometry of C1 at a size that streams from HBM (4k tokens, a
# 16-token patch at the end; the decode step is in its next_rows) -- the short-patch path of north_star at head_dim 64
D64 = synth.GraftConfig("D64-4k", 32, 32, 32, 64, 16, 1e4, 64, 128, 1024, 8192, 1, 6, 6, 4096, holes=((-1, 16),))
# likewise for head_dim 256 (R27; Gemma-2-9B geometry: 42 layers, 16 q / 8 kv heads): 4k tokens,
# a 16-token hole mid-cache and 48 tokens at the end in one call (R = 128 rows per kv head)
D256 = synth.GraftConfig("D256-4k", 42, 16, 8, 256, 16, 1e4, 64, 128, 1024, 8192, 1, 6, 6, 4096, holes=((2, 16), (-1, 48)))
BENCH_CONFIGS = dict(synth.CONFIGS, D64=D64, D256=D256)


def _peaks_file():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return json.load(f)
    except Exception:
        return None


def peaks():
    p = _peaks_file()
    if p and "hbm_gbs" in p:
        return float(p["hbm_gbs"]), "measured (MEASURED_PEAKS.json, torch copy_ read+write)"
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def tensor_peak():
    p = _peaks_file()
    if p and "bf16_tflops_sustained" in p:
        return float(p["bf16_tflops_sustained"]), "measured (MEASURED_PEAKS.json, sustained bf16 matmul)"
    return FALLBACK_BF16_SUSTAINED, "fallback (B200_PROFILING.md, sustained)"


# --------------------------------------------------------------------------------------------------
# algorithmic bytes
# --------------------------------------------------------------------------------------------------
def stitch_bytes(cfg, wl, tasks=None) -> int:
    """every stitched K/V byte is read once and written once: T_stitched * L * Hkv * D * 2 B * 2 (K,V) * 2 (r+w)."""
    tasks = wl.tasks if tasks is None else tasks
    return int(sum(n for t in tasks for (_, _, n, _) in t.entries)) * cfg.kv_bytes_per_token * 2


def attn_bytes(cfg, wl, tasks=None) -> int:
    """visible K+V read once per kv head: sum over tasks of L * kv_len * Hkv * D * 4 B (q/out/partials < 1 %)."""
    tasks = wl.tasks if tasks is None else tasks
    return int(sum(cfg.n_layers * (int(t.positions[-1]) + 1) * cfg.n_kv_heads * cfg.head_dim * 4 for t in tasks))


def attn_flops(cfg, wl, tasks=None) -> int:
    """Q K^T and P V over the visible cache only: per layer, q head and patch token i, 4 * D * (p_i + 1) flops."""
    tasks = wl.tasks if tasks is None else tasks
    vis = sum(int((np.asarray(t.positions, np.int64) + 1).sum()) for t in tasks)
    return 4 * cfg.head_dim * cfg.n_layers * cfg.n_q_heads * vis


def attn_rows(cfg, wl, tasks=None) -> int:
    """largest R = n * G (query rows per kv head) of the batch: intensity of patch attention is R flop/B."""
    tasks = wl.tasks if tasks is None else tasks
    return max(len(t.positions) for t in tasks) * (cfg.n_q_heads // cfg.n_kv_heads)


def ncu_traffic():
    """dram__bytes_read.sum + dram__bytes_write.sum per launch, from the committed `ncu --set full` summaries:
    the newest profiles/r*_traffic.csv (columns: config, kernel, dram_bytes_per_launch, capture).  {} if none."""
    pdir = os.path.join(ROOT, "profiles")
    try:
        files = sorted(f for f in os.listdir(pdir) if f.endswith("_traffic.csv"))
    except OSError:
        return {}, None
    if not files:
        return {}, None
    out = {}
    with open(os.path.join(pdir, files[-1])) as f:
        for row in csv.DictReader(f):
            try:
                out.setdefault(row["config"], {})[row["kernel"]] = float(row["dram_bytes_per_launch"])
            except (KeyError, ValueError):
                continue
    return out, "profiles/" + files[-1]


# --------------------------------------------------------------------------------------------------
# clocks during the timed regions
# --------------------------------------------------------------------------------------------------
class ClockSampler:
    """SM clock, power and clock-event (throttle) reasons of one GPU, sampled for the whole run by a background thread
    and cut into windows afterwards, so that every timed region reports the samples that fall INSIDE it.
    Source: NVML (what nvidia-smi reads) polled every ~4 ms; if pynvml cannot be used, `nvidia-smi -lms 20` with the
    query of B200_PROFILING.md."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, cuda_index: int):
        self.index, self.rows, self.proc, self.thread = cuda_index, [], None, None
        self.source, self.sm_max, self._stop = None, None, False

    def start(self):
        try:
            import pynvml as N
            N.nvmlInit()
            h = None
            try:
                uuid = str(torch.cuda.get_device_properties(self.index).uuid)
                h = N.nvmlDeviceGetHandleByUUID(("GPU-" + uuid) if not uuid.startswith("GPU-") else uuid)
            except Exception:
                vis = os.environ.get("CUDA_VISIBLE_DEVICES", "")
                idx = int(vis.split(",")[self.index]) if vis and all(x.strip().isdigit() for x in vis.split(",")) else self.index
                h = N.nvmlDeviceGetHandleByIndex(idx)
            self.sm_max = float(N.nvmlDeviceGetMaxClockInfo(h, N.NVML_CLOCK_SM))
            masks = (("hw_slowdown", N.nvmlClocksEventReasonHwSlowdown), ("hw_thermal_slowdown", N.nvmlClocksEventReasonHwThermalSlowdown),
                     ("sw_thermal_slowdown", N.nvmlClocksEventReasonSwThermalSlowdown), ("sw_power_cap", N.nvmlClocksEventReasonSwPowerCap),
                     ("hw_power_brake_slowdown", N.nvmlClocksEventReasonHwPowerBrakeSlowdown))

            def loop():
                while not self._stop:
                    try:
                        sm = float(N.nvmlDeviceGetClockInfo(h, N.NVML_CLOCK_SM))
                        bits = int(N.nvmlDeviceGetCurrentClocksEventReasons(h))
                        pw = N.nvmlDeviceGetPowerUsage(h) / 1000.0
                        self.rows.append((time.time(), sm, [n for n, m in masks if bits & m], pw))
                    except Exception:
                        pass
                    time.sleep(0.004)

            N.nvmlDeviceGetClockInfo(h, N.NVML_CLOCK_SM)          # fail here, not in the thread
            self.source = "nvml (pynvml), ~4 ms period"
            self.thread = threading.Thread(target=loop, daemon=True)
            self.thread.start()
            return
        except Exception:
            pass
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "20", "-i", str(self.index)], stdout=subprocess.PIPE, text=True)
            self.source = "nvidia-smi -lms 20"
            threading.Thread(target=self._read_smi, daemon=True).start()
        except Exception:
            self.proc = None

    def _read_smi(self):
        for line in self.proc.stdout:
            r = [x.strip() for x in line.split(",")]
            try:
                reasons = [n for n, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[5:9])
                           if v.lower().startswith("active")]
                self.sm_max = float(r[2])
                self.rows.append((time.time(), float(r[1]), reasons, float(r[3])))
            except Exception:
                continue

    def window(self, t0: float, t1: float) -> dict:
        if self.source is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no clock source (pynvml and nvidia-smi unavailable)"], "samples": 0}
        inside = [r for r in list(self.rows) if t0 <= r[0] <= t1]
        where = "timed region"
        if len(inside) < 3:
            inside = [r for r in list(self.rows) if t0 - 0.1 <= r[0] <= t1 + 0.1]
            where = "timed region +- 0.1 s (fewer than 3 samples fell inside)"
        sm = [r[1] for r in inside]
        reasons = sorted({x for r in inside for x in r[2]})
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_min_mhz": float(np.min(sm)) if sm else None,
                "sm_max_mhz": self.sm_max, "power_w_max": float(max(r[3] for r in inside)) if inside else None,
                "reasons": reasons, "samples": len(sm), "window": where, "source": self.source}

    def stop(self):
        self._stop = True
        if self.proc is not None:
            self.proc.terminate()


# --------------------------------------------------------------------------------------------------
# the CUDA arm: library, inputs, one timed region
# --------------------------------------------------------------------------------------------------
def build_library(cfg, wl, seed, device_index, on_segment=None, kv_heads=None, tasks=None, extra=True):
    """The library exactly as the timed run uses it.  `on_segment(s, k, v)` lets the full-size parity tests keep
    slices of the device-generated segments for the oracle.  `kv_heads = (begin, end)`: head-parallel shard -- `cfg`
    is then the sharded configuration and every segment is cut to those kv heads after generation (same bits as the
    unsharded run).  `tasks`: the tasks this rank grafts (task-parallel shard); default all."""
    from paper_2606_13097_b200 import binding
    tasks = wl.tasks if tasks is None else tasks
    total_pages = sum(-(-t.capacity // cfg.page_size) for t in tasks)
    seg_tokens = int(wl.seg_lens.sum())
    n_fp8 = 0
    if extra:
        # + EXTRACT_TOKENS of arena and + half a task of pages: room for the NEXT-row measurements (segment extraction,
        # copy-on-shift, fp8 copies of task 0's segments); none changes what the graft step itself touches
        used0 = sorted({s for (s, _, _, _) in tasks[0].entries})
        n_fp8 = len(used0)
        seg_tokens += EXTRACT_TOKENS + int(sum(int(wl.seg_lens[s]) for s in used0)) * 5 // 8 + 16 * n_fp8
        total_pages += max(-(-t.capacity // cfg.page_size) for t in tasks) // 2 + 8
    full = wl.cfg
    lib = binding.FcgLibrary(n_layers=cfg.n_layers, n_q_heads=cfg.n_q_heads, n_kv_heads=cfg.n_kv_heads,
                             head_dim=cfg.head_dim, page_size=cfg.page_size, rope_base=cfg.rope_base,
                             max_segments=full.n_segments + 1 + n_fp8, max_tasks=max(max(t.task_id for t in tasks) + 1, 1),
                             max_task_tokens=max(t.capacity for t in tasks), n_pages=total_pages + 16,
                             workspace_bytes=2 << 30, segment_tokens=seg_tokens, device=device_index,
                             host_tier_tokens=(int(wl.seg_lens[tasks[0].entries[0][0]]) + 16) if extra else 0)
    dev = torch.device("cuda", device_index)
    gen_cfg = synth.scaled(full, page_size=cfg.page_size)
    for s in range(full.n_segments):
        k, v = synth.segment_kv(gen_cfg, s, int(wl.seg_lens[s]), seed, dev)
        if kv_heads is not None:
            k, v = k[:, kv_heads[0]:kv_heads[1]].contiguous(), v[:, kv_heads[0]:kv_heads[1]].contiguous()
        sid = lib.segment_register(k, v, int(wl.orig_starts[s]))
        assert sid == s
        if on_segment is not None:
            on_segment(s, k, v)
        del k, v
    torch.cuda.synchronize(dev)
    return lib


def plans_for(wl, tasks=None):
    tasks = wl.tasks if tasks is None else tasks
    return [{"task_id": t.task_id, "entries": t.entries, "holes": t.holes, "capacity_tokens": t.capacity} for t in tasks]


def patch_inputs(full_cfg, tasks, seed, dev, q_heads=None, kv_heads=None):
    """q, k, v of every task's patch, concatenated along the token axis (the layout fcg_patch_batch takes); head-parallel
    shards cut the same tensors to their heads."""
    qs = [synth.patch_qkv(full_cfg, t.task_id, len(t.positions), seed, dev) for t in tasks]
    q = torch.cat([x[0] for x in qs], dim=1)
    k = torch.cat([x[1] for x in qs], dim=1)
    v = torch.cat([x[2] for x in qs], dim=1)
    if q_heads is not None:
        q, k, v = q[:, :, q_heads[0]:q_heads[1]], k[:, :, kv_heads[0]:kv_heads[1]], v[:, :, kv_heads[0]:kv_heads[1]]
    return q.contiguous(), k.contiguous(), v.contiguous()


class Dist:
    """rank / world and the two collectives the bench needs (barrier, max over ranks); a no-op at world 1."""

    def __init__(self, args):
        self.rank = int(os.environ.get("RANK", "0"))
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        self.local = 0 if args.devices == "same" else int(os.environ.get("LOCAL_RANK", "0"))
        self.backend = None
        if self.world > 1:
            import torch.distributed as dist
            self.backend = "gloo" if args.devices == "same" else "nccl"
            if self.backend == "nccl":
                dist.init_process_group("nccl", device_id=torch.device("cuda", self.local))
            else:
                dist.init_process_group("gloo")
        torch.cuda.set_device(self.local)
        self.dev = torch.device("cuda", self.local)

    def barrier(self):
        torch.cuda.synchronize(self.dev)
        if self.world > 1:
            import torch.distributed as dist
            dist.barrier()
        torch.cuda.synchronize(self.dev)

    def max(self, x: float) -> float:
        if self.world == 1:
            return float(x)
        return shard.max_over_ranks(x, device=self.dev if self.backend == "nccl" else "cpu")

    def sum(self, x: float) -> float:
        if self.world == 1:
            return float(x)
        import torch.distributed as dist
        t = torch.tensor([float(x)], dtype=torch.float64, device=self.dev if self.backend == "nccl" else "cpu")
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
        return float(t.item())

    def close(self):
        if self.world > 1:
            import torch.distributed as dist
            dist.barrier()
            dist.destroy_process_group()


def time_region(lib, plans, ids, npt, pos, q, k, v, out, steps, warmup, D: Dist):
    """W warm-up steps, barrier + synchronize, EXACTLY `steps` timed steps bracketed by CUDA events on the launching
    stream (torch's current stream, which the binding passes to the library), barrier + synchronize."""
    live = [False]

    def step(ev=None):
        if live[0]:
            for tid in ids:
                lib.task_release(tid)
        if ev:
            ev[0].record()
        lib.stitch(plans)
        live[0] = True
        if ev:
            ev[1].record()
        if len(ids) == 1:
            lib.patch(ids[0], 0, q, k, v, pos, out)
        else:
            lib.patch_batch(ids, npt, 0, q, k, v, pos, out)
        if ev:
            ev[2].record()

    for _ in range(warmup):
        step()
    D.barrier()
    s0 = lib.stats()
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(steps)]
    t_begin, t_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    w0 = time.time()
    t_begin.record()
    for i in range(steps):
        step(evs[i])
    t_end.record()
    D.barrier()
    w1 = time.time()
    s1 = lib.stats()
    total_ms = D.max(t_begin.elapsed_time(t_end))
    return {"ms_per_step": total_ms / steps, "steps": steps,
            "stitch_ms": [e[0].elapsed_time(e[1]) for e in evs], "patch_ms": [e[1].elapsed_time(e[2]) for e in evs],
            "launches": int(sum(s1[f] - s0[f] for f in s1 if f.endswith("_launches"))), "wall": (w0, w1), "stats": s1}


def time_e2e(lib, plans, ids, npt, pos, q, k, v, out, steps, warmup, D: Dist):
    """the same step through the C ABI with HOST buffers: H2D of q/k/v and D2H of out inside the timed region, the host
    reads `out` every step (synchronize).  Returns (ms per step, h2d bytes, d2h bytes)."""
    qh, kh, vh = [x.cpu().contiguous().pin_memory() for x in (q, k, v)]
    oh = torch.empty_like(qh).pin_memory()
    single = len(ids) == 1

    def step_host():
        for tid in ids:
            lib.task_release(tid)
        lib.stitch(plans)
        if single:
            lib.patch_host(ids[0], 0, qh, kh, vh, pos, oh)
        else:
            lib.patch_batch_host(ids, npt, 0, qh, kh, vh, pos, oh)
        torch.cuda.synchronize(D.dev)          # the caller reads `out` on the host every step

    for _ in range(min(warmup, 3)):
        step_host()
    D.barrier()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    for _ in range(steps):
        step_host()
    b.record()
    D.barrier()
    ms = D.max(a.elapsed_time(b) / steps)
    # the host call patches in layer groups, so its KV-split choice (and with it the summation order) may differ from
    # the one-call device step: same result within the attention tolerance, not necessarily the same bits
    assert torch.allclose(oh.float(), out.cpu().float(), rtol=2e-2, atol=1e-2), "host-buffer call and device call disagree"
    return ms, int(qh.numel() + kh.numel() + vh.numel()) * 2, int(oh.numel()) * 2


def rooflines(cfg, wl, tasks, timing, traffic, name):
    """stitch (HBM) and patch-attention (HBM below R ~ 250 rows per kv head, bf16 tensor peak above) rooflines of one
    timed region, from the mean CUDA-event durations of its steps."""
    sb, ab = stitch_bytes(cfg, wl, tasks), attn_bytes(cfg, wl, tasks)
    af, rows = attn_flops(cfg, wl, tasks), attn_rows(cfg, wl, tasks)
    peak, peak_src = peaks()
    st_s, at_s = float(np.mean(timing["stitch_ms"])) * 1e-3, float(np.mean(timing["patch_ms"])) * 1e-3
    tr = traffic.get(name, {})
    stitch = {"kernel": "stitch_kernel (fused gather + RoPE-shift)", "bound": "hbm", "achieved": sb / st_s / 1e9, "peak": peak,
              "unit": "GB/s", "frac": sb / st_s / 1e9 / peak, "peak_source": peak_src, "frac_of_8TBps": sb / st_s / 1e9 / 8000.0,
              "traffic": tr.get("stitch")}
    # intensity of the whole call in flop per K/V byte (= R for a single task; a mixed batch like C4 averages its tasks):
    # tensor-bound from ~250 flop/B (sustained bf16 peak / measured HBM peak), HBM-bound below
    if af / max(ab, 1) >= 250:
        tpeak, tsrc = tensor_peak()
        attn = {"kernel": "attn_tc_kernel (tcgen05 / TMEM)", "bound": "tensor", "achieved": af / at_s / 1e12, "peak": tpeak, "unit": "TFLOP/s",
                "frac": af / at_s / 1e12 / tpeak, "peak_source": tsrc, "rows_per_kv_head": rows, "flop_per_byte": af / max(ab, 1),
                "hbm_GBps": ab / at_s / 1e9, "hbm_frac": ab / at_s / 1e9 / peak}
    else:
        attn = {"kernel": "attn_tc_kernel (tcgen05 / TMEM)" if timing["stats"]["last_attn_path"] == 2 else "attn_split_kernel (mma.sync split-KV)",
                "bound": "hbm", "achieved": ab / at_s / 1e9, "peak": peak, "unit": "GB/s", "frac": ab / at_s / 1e9 / peak,
                "frac_of_8TBps": ab / at_s / 1e9 / 8000.0, "rows_per_kv_head": rows, "flop_per_byte": af / max(ab, 1),
                "TFLOPs": af / at_s / 1e12}
    attn["traffic"] = tr.get("attn")
    attn["note"] = "timed as scatter + attention (+ combine); scatter is ~1 % of it"
    return stitch, attn, sb, ab, af


def describe(cfg, name, wl, tasks, seed):
    return (f"{cfg.name} ({name}): L={cfg.n_layers} Hq={cfg.n_q_heads} Hkv={cfg.n_kv_heads} D={cfg.head_dim} page={cfg.page_size} "
            f"base={cfg.rope_base:g}; library {wl.cfg.n_segments} segments ({int(wl.seg_lens.sum())} tokens); {len(tasks)} task(s), "
            f"{int(sum(n for t in tasks for (_, _, n, _) in t.entries))} stitched + {int(sum(len(t.positions) for t in tasks))} patch tokens; "
            f"layout seed {seed}")


def measure_config(args, name, seed, D: Dist, sampler, traffic, steps, *, full, shard_mode="none"):
    """One configuration on this rank's shard: build the library, time `steps` graft steps; `full` adds the end-to-end
    leg and (rank 0) the NEXT rows.  Returns the per-config record (rank 0 decides what to print)."""
    cfg_full = BENCH_CONFIGS[name]
    if args.page_size:
        cfg_full = synth.scaled(cfg_full, page_size=args.page_size)
    kv_heads = q_heads = None
    cfg = cfg_full
    scaling = "weak"
    if shard_mode == "weak" and D.world > 1:
        # 32 x N independent tasks over one shared library, balanced over the ranks longest-first
        wl = synth.make_workload(synth.scaled(cfg_full, n_tasks=cfg_full.n_tasks * D.world), seed)
        mine, _ = shard.rank_workload(wl, D.rank, D.world, cfg.kv_bytes_per_token)
        tasks = [wl.tasks[i] for i in mine]
    elif shard_mode == "task" and D.world > 1:
        wl = synth.make_workload(cfg_full, seed)
        mine, _ = shard.rank_workload(wl, D.rank, D.world, cfg.kv_bytes_per_token)
        tasks = [wl.tasks[i] for i in mine]
        scaling = "strong"
    elif shard_mode == "head" and D.world > 1:
        wl = synth.make_workload(cfg_full, seed)
        tasks = wl.tasks
        cfg = shard.head_sharded_config(cfg_full, D.rank, D.world)
        kv_heads = shard.kv_head_range(cfg_full.n_kv_heads, D.rank, D.world)
        q_heads = shard.q_head_range(cfg_full.n_q_heads, cfg_full.n_kv_heads, D.rank, D.world)
        scaling = "strong"
    else:
        wl = synth.make_workload(cfg_full, seed)
        tasks = wl.tasks
    if not tasks:
        raise RuntimeError(f"rank {D.rank} has no task of {name} (world {D.world} > tasks)")
    lib = build_library(cfg, wl, seed, D.local, kv_heads=kv_heads, tasks=tasks, extra=full)
    try:
        plans = plans_for(wl, tasks)
        ids = [t.task_id for t in tasks]
        npt = [len(t.positions) for t in tasks]
        pos = np.concatenate([t.positions for t in tasks]).astype(np.int32)
        q, k, v = patch_inputs(synth.scaled(cfg_full, page_size=cfg.page_size), tasks, seed, D.dev, q_heads, kv_heads)
        out = torch.empty_like(q)
        timing = time_region(lib, plans, ids, npt, pos, q, k, v, out, steps, args.warmup, D)
        stitch_roof, attn_roof, sb, ab, af = rooflines(cfg, wl, tasks, timing, traffic, name)
        # whole-job units: every rank's bytes (summed) over the max-over-ranks time
        job_bytes = D.sum(sb + ab)
        ms = timing["ms_per_step"]
        rec = {
            "workload": describe(cfg, name, wl, tasks, seed) + (f"; rank 0 of {D.world}, shard = {shard_mode}" if D.world > 1 else ""),
            "ms_per_step": ms, "steps": steps, "value_GBps": job_bytes / (ms * 1e-3) / 1e9,
            "stitch_ms": float(np.mean(timing["stitch_ms"])), "stitch_ms_min": float(np.min(timing["stitch_ms"])),
            "stitch_ms_median": float(np.median(timing["stitch_ms"])),
            "patch_ms": float(np.mean(timing["patch_ms"])), "patch_ms_min": float(np.min(timing["patch_ms"])),
            "patch_ms_median": float(np.median(timing["patch_ms"])),
            "stitch_bytes": sb, "attn_bytes": ab, "attn_flops": af,
            "attn_path": timing["stats"]["last_attn_path"], "attn_splits": timing["stats"]["last_attn_splits"],
            "gpu_launches": timing["launches"], "scaling": scaling,
            "l2": "inputs larger than L2 (each step streams >= 1 GiB; no flush needed)" if sb > 4 * 126e6
            else "working set fits L2: latency only, no roofline claim",
            "roofline": dict(stitch_roof, patch_attention=attn_roof),
            "clocks": sampler.window(*timing["wall"]) if sampler else None,
            "_job_bytes": job_bytes,
        }
        if sb <= 4 * 126e6:
            rec["roofline"] = None
        if full:
            e_ms, h2d, d2h = time_e2e(lib, plans, ids, npt, pos, q, k, v, out, max(3, min(steps, 10)), args.warmup, D)
            rec["e2e"] = {"value": job_bytes / (e_ms * 1e-3) / 1e9, "unit": UNIT, "ms_per_step": e_ms,
                          "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h}
            if D.rank == 0 and not args.no_next and shard_mode in ("none", "replica"):
                try:
                    rec["next_rows"] = time_next_rows(lib, cfg, wl, seed, D.dev)
                except Exception as e:       # never lose the main line to an extra
                    rec["next_rows"] = {"error": repr(e)}
            if D.rank == 0 and name == "C5" and not args.no_prefill_compare and shard_mode in ("none", "replica"):
                try:
                    pc = time_prefill_compare(lib, cfg, wl, seed, D.dev)
                    pc["graft_ms"] = ms
                    pc["prefill_attention_over_graft"] = pc["own_kernel_ms_all_layers"] / ms
                    rec["prefill_compare"] = pc
                except Exception as e:
                    rec["prefill_compare"] = {"error": repr(e)}
        if D.world > 1 and shard_mode in ("head", "task", "weak") and out.numel() * 2 * D.world <= (1 << 30) and D.backend == "nccl":
            # results are exchanged only here, outside every timed region (shard.py); head shards concatenate along the
            # head axis, task shards are put back in task order
            if shard_mode == "head":
                whole = shard.gather_head_outputs(out)
                rec["gathered_out_shape"] = list(whole.shape)
                del whole
        return rec, lib, (cfg, wl, tasks)
    except Exception:
        lib.close()
        raise


def time_next_rows(lib, cfg, wl, seed, dev, iters=5):
    """SURVEY.md 8(f) NEXT rows, timed on task 0 of the stitched workload after the main measurement (CUDA events,
    2 warm-ups): suffix re-graft by -16 / +16 tokens (fcg_task_shift), extraction of EXTRACT_TOKENS tokens into the
    library (fcg_segment_extract), one decode step (fcg_patch, n = 1, R = G) over the whole cache, the one-call-per-layer
    pattern (plain calls, a patch plan, and the plan captured into one CUDA graph) and the two-tier moves."""
    t = wl.tasks[0]
    cap = t.capacity
    mid = (cap // 2) & ~15
    n_shift = cap - mid - 16
    n_ext = min(EXTRACT_TOKENS, mid)
    q, k, v = synth.patch_qkv(cfg, t.task_id, 1, seed + 100, dev)
    out = torch.empty_like(q)
    pos = np.asarray([cap - 1], np.int32)

    def shift_pair():
        lib.task_shift(t.task_id, mid + 16, n_shift, mid)
        lib.task_shift(t.task_id, mid, n_shift, mid + 16)

    def extract():
        lib.segment_release(lib.segment_extract(t.task_id, 0, n_ext, 0))

    def decode():
        lib.patch(t.task_id, 0, q, k, v, pos, out)

    kr, vr = synth.segment_kv(cfg, 0, n_ext, seed + 200, dev)      # S1: a caller's K/V copied into the library

    def register():
        lib.segment_release(lib.segment_register(kr, vr, 0))

    def timed_loop(fn, n=iters, warm=2):
        for _ in range(warm):
            fn()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize(dev)
        t0 = time.perf_counter()
        a.record()
        for _ in range(n):
            fn()
        b.record()
        t1 = time.perf_counter()
        torch.cuda.synchronize(dev)
        return a.elapsed_time(b) / n, (t1 - t0) * 1e3 / n

    def release0():
        """task 0 goes away if it is live (other tasks of a batched workload stay)"""
        try:
            lib.task_release(t.task_id)
        except Exception:
            pass

    res = {}
    # the call pattern of a model that patches layer by layer: L calls of one layer each (task 0's own patch tokens)
    try:
        qp, kp, vp = synth.patch_qkv(cfg, t.task_id, len(t.positions), seed, dev)
        op = torch.empty_like(qp)
        views = [(qp[l:l + 1], kp[l:l + 1], vp[l:l + 1], op[l:l + 1]) for l in range(cfg.n_layers)]

        def per_layer():
            for l, (a_, b_, c_, d_) in enumerate(views):
                lib.patch(t.task_id, l, a_, b_, c_, t.positions, d_)

        ms, host = timed_loop(per_layer)
        res["patch_one_call_per_layer"] = {"ms": ms, "host_enqueue_ms": host, "calls": cfg.n_layers, "splits": lib.stats()["last_attn_splits"],
                                           "note": "same patch as the timed step, issued as one fcg_patch per layer"}
        plan = lib.patch_plan_create([t.task_id], [len(t.positions)], t.positions, 1)

        def per_layer_planned():
            for l, (a_, b_, c_, d_) in enumerate(views):
                lib.patch_planned(plan, l, a_, b_, c_, d_)

        ms, host = timed_loop(per_layer_planned)
        res["patch_one_call_per_layer_planned"] = {"ms": ms, "host_enqueue_ms": host, "calls": cfg.n_layers,
                                                   "note": "fcg_patch_plan_create once, then one fcg_patch_planned per layer (launches only)"}
        side = torch.cuda.Stream(device=dev)
        side.wait_stream(torch.cuda.current_stream(dev))
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=side):
            per_layer_planned()
        ms, host = timed_loop(g.replay)
        res["patch_one_call_per_layer_graph"] = {"ms": ms, "host_enqueue_ms": host, "calls": 1,
                                                 "note": f"the {cfg.n_layers} planned per-layer calls captured into one CUDA graph, one replay per step"}
        del g
        # layers are independent: inside the capture the per-layer calls are forked over 8 streams (their split-KV
        # partials live in per-layer slots), so the launch latencies of one layer hide behind the kernels of the others
        # ... and the plan's KV-split choice is made for n_lanes layers in flight (no split, no combine kernel needed)
        n_lanes = 8
        lib.patch_plan_destroy(plan)
        plan = lib.patch_plan_create([t.task_id], [len(t.positions)], t.positions, min(n_lanes, cfg.n_layers))
        lanes = [side] + [torch.cuda.Stream(device=dev) for _ in range(n_lanes - 1)]
        g4 = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g4, stream=side):
            fork = torch.cuda.Event()
            fork.record(side)
            for st_ in lanes[1:]:
                st_.wait_event(fork)
            for l, (a_, b_, c_, d_) in enumerate(views):
                lib.patch_planned(plan, l, a_, b_, c_, d_, stream=lanes[l % n_lanes])
            for st_ in lanes[1:]:
                ev = torch.cuda.Event()
                ev.record(st_)
                side.wait_event(ev)
        ms, host = timed_loop(g4.replay)
        res["patch_one_call_per_layer_graph_8_lanes"] = {"ms": ms, "host_enqueue_ms": host, "calls": 1,
                                                         "note": "the same per-layer calls forked round-robin over 8 captured streams, plan made for 8 layers in flight"}
        del g4
        lib.patch_plan_destroy(plan)
        del qp, kp, vp, op, views
    except Exception as e:
        res["patch_one_call_per_layer_error"] = repr(e)
    per_tok = cfg.kv_bytes_per_token
    for name, fn, nbytes in (("decode_step", decode, cfg.n_layers * cap * cfg.n_kv_heads * cfg.head_dim * 4),
                             ("segment_register", register, n_ext * per_tok * 2),
                             ("segment_extract", extract, n_ext * per_tok * 2),
                             ("task_shift", shift_pair, 2 * n_shift * per_tok * 2)):
        ms, _ = timed_loop(fn)
        res[name] = {"ms": ms, "GBps": nbytes / (ms * 1e-3) / 1e9, "bytes": int(nbytes)}
    # NEXT-3 two-tier residency: one library segment to the pinned host tier and back (copy engine), and a stitch
    # that reads it in place from the host tier (zero-copy over the host link)
    seg = int(t.entries[0][0])
    n_seg = int(wl.seg_lens[seg])
    seg_bytes = n_seg * per_tok
    try:
        release0()
        plan = [{"task_id": t.task_id, "entries": [(seg, 0, n_seg, 0)], "holes": [], "capacity_tokens": n_seg}]

        def timed(fn, before=None, n=3):
            ms = []
            for _ in range(n + 1):
                if before:
                    before()
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                torch.cuda.synchronize(dev)
                a.record()
                fn()
                b.record()
                torch.cuda.synchronize(dev)
                ms.append(a.elapsed_time(b))
            return float(np.mean(ms[1:]))

        off_ms = timed(lambda: lib.segment_offload(seg), before=lambda: lib.segment_prefetch(seg))
        pre_ms = timed(lambda: lib.segment_prefetch(seg), before=lambda: lib.segment_offload(seg))
        lib.segment_offload(seg)
        host_ms = timed(lambda: lib.stitch(plan), before=release0)
        release0()
        lib.segment_prefetch(seg)
        # NEXT-3 overlap: task 0's real plan with its first segment in the host tier -- read in place (fcg_stitch) vs
        # copied back by the copy engine while the resident entries are stitched (fcg_stitch_prefetch)
        try:
            plan0 = [{"task_id": t.task_id, "entries": t.entries, "holes": t.holes, "capacity_tokens": t.capacity}]
            def before():
                release0()
                lib.segment_offload(seg)

            inplace_ms = timed(lambda: lib.stitch(plan0), before=before)
            overlap_ms = timed(lambda: lib.stitch_prefetch(plan0), before=before)
            release0()
            res["stitch_prefetch_overlap"] = {"ms": overlap_ms, "in_place_ms": inplace_ms, "offloaded_bytes": int(seg_bytes),
                                              "offloaded_GBps": seg_bytes / (overlap_ms * 1e-3) / 1e9,
                                              "note": f"task 0's plan ({sum(n for (_, _, n, _) in t.entries)} tokens) with one {n_seg}-token segment offloaded: "
                                                      "fcg_stitch_prefetch (copy engine + overlapped stitch of the resident entries; the segment ends up "
                                                      "resident) vs fcg_stitch reading it in place over the host link"}
        except Exception as e:
            res["stitch_prefetch_overlap"] = {"error": repr(e)}
        res["segment_offload"] = {"ms": off_ms, "GBps": seg_bytes / (off_ms * 1e-3) / 1e9, "bytes": int(seg_bytes)}
        res["segment_prefetch"] = {"ms": pre_ms, "GBps": seg_bytes / (pre_ms * 1e-3) / 1e9, "bytes": int(seg_bytes)}
        res["stitch_from_host_tier"] = {"ms": host_ms, "GBps": seg_bytes / (host_ms * 1e-3) / 1e9, "bytes": int(seg_bytes),
                                        "note": f"{n_seg}-token segment read in place from pinned host memory (bytes = one-way)"}
    except Exception as e:
        res["two_tier"] = {"error": repr(e)}
    # NEXT-4 fp8 library storage (R26): task 0's segments once more as fp8 segments, the same plan stitched from them;
    # algorithmic bytes per stitched token = L * Hkv * (2 D + 2 read + 4 D written) instead of L * Hkv * 8 D
    try:
        used0 = sorted({s for (s, _, _, _) in t.entries})
        gen_cfg = synth.scaled(wl.cfg, page_size=cfg.page_size)
        fp8_id = {}
        for s_ in used0:
            k8, v8 = synth.segment_kv(gen_cfg, s_, int(wl.seg_lens[s_]), seed, dev)
            if k8.shape[1] != cfg.n_kv_heads:
                raise RuntimeError("head-sharded library: fp8 row skipped")
            fp8_id[s_] = lib.segment_register_fp8(k8, v8, int(wl.orig_starts[s_]))
            del k8, v8
        n_st = int(sum(n for (_, _, n, _) in t.entries))
        plan16 = [{"task_id": t.task_id, "entries": t.entries, "holes": t.holes, "capacity_tokens": t.capacity}]
        plan8 = [{"task_id": t.task_id, "entries": [(fp8_id[s_], b_, n_, d_) for (s_, b_, n_, d_) in t.entries], "holes": t.holes,
                  "capacity_tokens": t.capacity}]

        def restitch(pl_):
            def f():
                release0()
                lib.stitch(pl_)
            return f

        ms16, _ = timed_loop(restitch(plan16))
        ms8, _ = timed_loop(restitch(plan8))
        release0()
        b16 = n_st * cfg.n_layers * cfg.n_kv_heads * cfg.head_dim * 8
        b8 = n_st * cfg.n_layers * cfg.n_kv_heads * (cfg.head_dim * 6 + 2)
        fmt, nb8 = lib.segment_storage(fp8_id[used0[0]])
        _, nb16 = lib.segment_storage(used0[0])
        res["stitch_fp8"] = {"ms": ms8, "GBps": b8 / (ms8 * 1e-3) / 1e9, "bytes": int(b8), "bf16_same_plan_ms": ms16,
                             "bf16_same_plan_GBps": b16 / (ms16 * 1e-3) / 1e9, "stored_bytes_ratio": nb8 / nb16,
                             "note": f"task 0 ({n_st} tokens) stitched from e4m3 segments (de-quantise -> rotate -> bf16 pages) vs from bf16 segments"}
        for s_ in used0:
            lib.segment_release(fp8_id[s_])
    except Exception as e:
        res["stitch_fp8"] = {"error": repr(e)}
    res["task_shift"]["note"] = f"two moves of {n_shift} tokens (-16, +16) per iteration"
    res["segment_extract"]["note"] = f"{n_ext} tokens un-rotated to orig_start 0"
    res["segment_register"]["note"] = f"S1: {n_ext} tokens copied into the library (read + write)"
    res["decode_step"]["note"] = f"n = 1 at position {cap - 1}, R = {cfg.n_q_heads // cfg.n_kv_heads} rows per kv head"
    return res


def time_prefill_compare(lib, cfg, wl, seed, dev, layers_per_call=4):
    """BASELINE.json configs[4]: "compare graft time to causal attention prefill over the same 32k tokens".
    Prefill attention = the same fcg_patch kernel with every position of a fresh task as a patch token (an empty cache
    plus one patch is causal self-attention, DESIGN.md pin P12); timed for `layers_per_call` layers and scaled to all
    layers (every layer does identical work).  The projections / MLP a real prefill also pays are NOT included, so
    the ratio understates what grafting saves.  torch SDPA on the same shapes is quoted as library context."""
    t = wl.tasks[0]
    T_ = t.capacity
    try:
        lib.task_release(t.task_id)          # live unless the NEXT-row timings already released it
    except Exception:
        pass
    lib.stitch([{"task_id": t.task_id, "entries": [], "holes": [(0, T_)], "capacity_tokens": T_}])
    sub = synth.scaled(cfg, n_layers=layers_per_call)
    q, k, v = synth.patch_qkv(sub, t.task_id, T_, seed + 7, dev)
    out = torch.empty_like(q)
    pos = np.arange(T_, dtype=np.int32)
    ms = []
    for _ in range(3):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize(dev)
        a.record()
        lib.patch(t.task_id, 0, q, k, v, pos, out)
        b.record()
        torch.cuda.synchronize(dev)
        ms.append(a.elapsed_time(b))
    own_ms = float(np.min(ms[1:])) * cfg.n_layers / layers_per_call
    flops = 4 * cfg.head_dim * cfg.n_q_heads * cfg.n_layers * (T_ * (T_ + 1) // 2)
    res = {"tokens": T_, "own_kernel_ms_all_layers": own_ms, "own_kernel_TFLOPs": flops / (own_ms * 1e-3) / 1e12,
           "timed_layers": layers_per_call, "flops_all_layers": int(flops)}
    try:
        import torch.nn.functional as F
        qs = q[0].permute(1, 0, 2).unsqueeze(0).contiguous()          # [1][Hq][T][D]
        ks = k[0].permute(1, 0, 2).unsqueeze(0).contiguous()
        vs = v[0].permute(1, 0, 2).unsqueeze(0).contiguous()
        sm = []
        for _ in range(3):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize(dev)
            a.record()
            F.scaled_dot_product_attention(qs, ks, vs, is_causal=True, enable_gqa=True)
            b.record()
            torch.cuda.synchronize(dev)
            sm.append(a.elapsed_time(b))
        res["torch_sdpa_ms_all_layers"] = float(np.min(sm[1:])) * cfg.n_layers
        res["torch_sdpa_note"] = "library kernel, context only"
    except Exception as e:
        res["torch_sdpa_ms_all_layers"] = None
        res["torch_sdpa_error"] = repr(e)
    lib.task_release(t.task_id)
    return res


def c1_latency(args, D, seed):
    """C1 (0.65 MiB, fits L2): launch-bound, latency only, no roofline claim."""
    cfg = synth.CONFIGS["C1"]
    wl = synth.make_workload(cfg, seed)
    lib = build_library(cfg, wl, seed, D.local, extra=False)
    try:
        t = wl.tasks[0]
        q, k, v = patch_inputs(cfg, wl.tasks, seed, D.dev)
        out = torch.empty_like(q)
        timing = time_region(lib, plans_for(wl), [t.task_id], [len(t.positions)], t.positions.astype(np.int32), q, k, v, out, 200, 5,
                             Dist.__new__(Dist)._solo(D))
        return {"workload": describe(cfg, "C1", wl, wl.tasks, seed), "ms_per_step": timing["ms_per_step"], "steps": 200,
                "stitch_ms_median": float(np.median(timing["stitch_ms"])), "patch_ms_median": float(np.median(timing["patch_ms"])),
                "attn_path": timing["stats"]["last_attn_path"], "note": "working set fits L2 and the step is launch-bound: latency only"}
    finally:
        lib.close()


def _solo(self, D):
    """a world-1 view of this rank (local measurements that the other ranks do not take part in)"""
    self.rank, self.world, self.local, self.backend, self.dev = 0, 1, D.local, None, D.dev
    return self


Dist._solo = _solo


def run_cuda(args):
    D = Dist(args)
    sampler = ClockSampler(D.local) if D.rank == 0 else None
    if sampler:
        sampler.start()
    traffic, traffic_src = ncu_traffic()
    single = args.config != "all"
    head_name = args.config if single else HEADLINE
    if D.world > 1:
        mode = args.shard if args.shard != "auto" else ("weak" if BENCH_CONFIGS[head_name].n_tasks > 1 else "head")
    else:
        mode = "none"
    if mode == "head" and BENCH_CONFIGS[head_name].n_kv_heads % D.world:
        mode = "replica"
    seeds = [int(s) for s in args.seeds.split(",") if s]
    configs = {}
    # ---- headline: EXACTLY K steps ----------------------------------------------------------------
    rec, lib, (cfg, wl, tasks) = measure_config(args, head_name, args.seed, D, sampler, traffic, args.steps, full=True, shard_mode=mode)
    res = {
        "metric": METRIC, "value": rec["value_GBps"], "unit": UNIT, "n_gpus": D.world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": rec["ms_per_step"], "higher_is_better": True, "scaling": rec["scaling"], "vs_baseline": None,
        "dtype": "bf16", "data": "synthetic",
        "config": {"workload": short_workload(head_name, cfg, len(tasks), int(sum(n for t in tasks for (_, _, n, _) in t.entries)),
                                              int(sum(len(t.positions) for t in tasks)), args.seed),
                   "workload_long": rec["workload"], "l2": rec["l2"], "stitch_ms": rec["stitch_ms"], "stitch_ms_min": rec["stitch_ms_min"],
                   "stitch_ms_median": rec["stitch_ms_median"], "patch_ms": rec["patch_ms"], "patch_ms_min": rec["patch_ms_min"],
                   "patch_ms_median": rec["patch_ms_median"], "stitch_bytes": rec["stitch_bytes"], "attn_bytes": rec["attn_bytes"],
                   "attn_flops": rec["attn_flops"], "attn_path": rec["attn_path"], "attn_splits": rec["attn_splits"],
                   "parallelism": {"none": "1 GPU", "replica": f"task-replica x{D.world}", "weak": f"task-parallel, {len(wl.tasks)} tasks LPT-balanced over {D.world} ranks",
                                   "task": f"task-parallel (strong), {D.world} ranks", "head": f"kv-head-parallel (strong), {D.world} ranks"}[mode],
                   "traffic_source": traffic_src},
        "gpu_launches": rec["gpu_launches"],
        "roofline": rec["roofline"],
        "clocks": rec["clocks"],
        "e2e": rec.get("e2e"),
    }
    if "next_rows" in rec:
        res["next_rows"] = rec["next_rows"]
    if "prefill_compare" in rec:
        res["prefill_compare"] = rec["prefill_compare"]
    if D.rank == 0 and D.world == 1 and not args.no_cpu_baseline:
        gen_cfg = synth.scaled(wl.cfg, page_size=cfg.page_size)
        res["cpu_baseline"] = cpu_baseline(cfg, wl, args.seed, lib_segments=lambda s: synth.segment_kv(gen_cfg, s, int(wl.seg_lens[s]), args.seed, D.dev))
    lib.close()
    del lib
    torch.cuda.empty_cache()
    configs[head_name] = {k: v for k, v in rec.items() if not k.startswith("_") and k not in ("next_rows",)}
    configs[head_name]["seeds"] = {str(args.seed): {"ms_per_step": rec["ms_per_step"], "stitch_ms": rec["stitch_ms"], "patch_ms": rec["patch_ms"]}}

    def region_steps(name):
        # sub-configurations: at least 20 steps and a region of >= ~0.12 s, so that the clock samples fall inside it
        est = {"C2": 1.0, "C3": 0.75, "C4": 8.0, "C5": 13.5, "D64": 0.5, "D256": 0.4}.get(name, 5.0)
        return int(max(20, args.steps, math.ceil(120.0 / est)))

    def other_seeds(name, mode_):
        out = {}
        for s in seeds:
            if s == args.seed:
                continue
            try:
                r, l, _ = measure_config(args, name, s, D, sampler, traffic, region_steps(name), full=False, shard_mode=mode_)
                l.close()
                del l
                torch.cuda.empty_cache()
                out[str(s)] = {"ms_per_step": r["ms_per_step"], "stitch_ms": r["stitch_ms"], "patch_ms": r["patch_ms"],
                               "stitch_frac": r["roofline"]["frac"] if r["roofline"] else None,
                               "patch_frac": r["roofline"]["patch_attention"]["frac"] if r["roofline"] else None}
            except Exception as e:
                out[str(s)] = {"error": repr(e)}
        return out

    if not args.no_seeds:
        configs[head_name]["seeds"].update(other_seeds(head_name, mode))
    # ---- the other configurations -------------------------------------------------------------------
    if not single:
        for name in ALL_CONFIGS:
            if name == head_name:
                continue
            c = synth.CONFIGS[name]
            m = "none" if D.world == 1 else ("head" if c.n_kv_heads % D.world == 0 else "replica")
            try:
                r, l, _ = measure_config(args, name, args.seed, D, sampler, traffic, region_steps(name), full=True, shard_mode=m)
                l.close()
                del l
                torch.cuda.empty_cache()
                if "prefill_compare" in r:
                    res["prefill_compare"] = r["prefill_compare"]
                configs[name] = {k: v for k, v in r.items() if not k.startswith("_")}
                configs[name]["seeds"] = {str(args.seed): {"ms_per_step": r["ms_per_step"], "stitch_ms": r["stitch_ms"], "patch_ms": r["patch_ms"]}}
                if not args.no_seeds:
                    configs[name]["seeds"].update(other_seeds(name, m))
            except Exception as e:
                configs[name] = {"error": repr(e)}
        if D.rank == 0:
            try:
                configs["C1"] = c1_latency(args, D, args.seed)
            except Exception as e:
                configs["C1"] = {"error": repr(e)}
        for extra in (("D64", "D256") if D.world == 1 else ()):
            try:
                r, l, _ = measure_config(args, extra, args.seed, D, sampler, traffic, region_steps(extra), full=True, shard_mode="none")
                l.close()
                del l
                torch.cuda.empty_cache()
                configs[extra] = {k: v for k, v in r.items() if not k.startswith("_")}
            except Exception as e:
                configs[extra] = {"error": repr(e)}
    res["configs"] = configs
    if sampler:
        sampler.stop()
    D.close()
    return res if D.rank == 0 else None


# --------------------------------------------------------------------------------------------------
# the line the driver reads: compact (< 4 KB), strict JSON, last on stdout.  Everything else goes on a DETAIL line.
# --------------------------------------------------------------------------------------------------
HEADLINE_MAX_BYTES = 4096


def _sig(x, digits=5):
    """numbers to `digits` significant digits (non-finite -> None: strict JSON), containers recursively"""
    if isinstance(x, bool) or x is None or isinstance(x, (int, str)):
        return x
    if isinstance(x, (float, np.floating)):
        x = float(x)
        if not math.isfinite(x):
            return None
        return float(f"{x:.{digits}g}")
    if isinstance(x, np.integer):
        return int(x)
    if isinstance(x, dict):
        return {k: _sig(v, digits) for k, v in x.items()}
    if isinstance(x, (list, tuple)):
        return [_sig(v, digits) for v in x]
    return str(x)


def _pick(d, keys, str_max=80):
    if not isinstance(d, dict):
        return None
    out = {}
    for k in keys:
        if k in d:
            v = d[k]
            out[k] = v[:str_max] if isinstance(v, str) else v
    return out


def short_workload(name, cfg, n_tasks, stitched, patched, seed):
    """<= 120 characters (the driver cuts `config.workload` there); the long description is on the DETAIL line"""
    return (f"{name}: L={cfg.n_layers} Hq={cfg.n_q_heads} Hkv={cfg.n_kv_heads} D={cfg.head_dim} page={cfg.page_size}; "
            f"{n_tasks} task(s), {stitched} stitched + {patched} patch tokens; seed {seed}")[:120]


def headline(res: dict) -> dict:
    """The compact record: the contract's keys, the dominant kernel's roofline (+ patch attention), cpu_baseline, clocks,
    e2e, C5's prefill comparison and six numbers per configuration.  `res` is the full record of run_cuda."""
    roof_keys = ("kernel", "bound", "achieved", "peak", "unit", "frac", "traffic", "frac_of_8TBps")
    cfg_in = res.get("config") or {}
    config = _pick(cfg_in, ("workload", "l2", "stitch_ms", "stitch_ms_min", "stitch_ms_median", "patch_ms", "patch_ms_min",
                            "patch_ms_median", "stitch_bytes", "attn_bytes", "attn_flops", "attn_path", "attn_splits", "parallelism"), 120)
    if "l2" in config:
        config["l2"] = config["l2"][:60]
    out = {k: res.get(k) for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                                   "vs_baseline", "dtype", "data", "gpu_launches")}
    out["config"] = config
    roof = res.get("roofline")
    if isinstance(roof, dict):
        r = _pick(roof, roof_keys, 60)
        r["peak_source"] = "MEASURED_PEAKS.json" if "MEASURED_PEAKS" in str(roof.get("peak_source")) else "fallback"
        pa = roof.get("patch_attention")
        if isinstance(pa, dict):
            r["patch_attention"] = _pick(pa, roof_keys + ("rows_per_kv_head", "hbm_GBps"), 60)
        out["roofline"] = r
    else:
        out["roofline"] = None
    cb = res.get("cpu_baseline")
    out["cpu_baseline"] = _pick(cb, ("value", "unit", "cores", "kind", "seconds", "sample"), 200) if cb else None
    out["clocks"] = _pick(res.get("clocks"), ("sm_mhz", "sm_min_mhz", "sm_max_mhz", "power_w_max", "reasons", "samples"))
    out["e2e"] = _pick(res.get("e2e"), ("value", "unit", "ms_per_step", "h2d_bytes_per_step", "d2h_bytes_per_step"))
    pc = res.get("prefill_compare")
    if isinstance(pc, dict):
        out["prefill_compare"] = _pick(pc, ("tokens", "graft_ms", "own_kernel_ms_all_layers", "torch_sdpa_ms_all_layers", "error"), 80)
        if pc.get("graft_ms") and pc.get("own_kernel_ms_all_layers"):
            out["prefill_compare"]["ratio"] = pc["own_kernel_ms_all_layers"] / pc["graft_ms"]
    summ = {}
    for name, c in (res.get("configs") or {}).items():
        if not isinstance(c, dict) or "error" in c:
            summ[name] = {"error": str((c or {}).get("error"))[:60]}
            continue
        roof_c = c.get("roofline") or {}
        pa_c = roof_c.get("patch_attention") or {}
        summ[name] = {"step_ms": c.get("ms_per_step"), "stitch_frac": roof_c.get("frac"), "patch_frac": pa_c.get("frac"),
                      "patch_bound": pa_c.get("bound"), "e2e_ms": (c.get("e2e") or {}).get("ms_per_step"),
                      "sm_mhz": (c.get("clocks") or {}).get("sm_mhz")}
    out["configs_summary"] = summ
    out["detail"] = "the full per-configuration record is the earlier stdout line that starts with DETAIL"
    out = _sig(out)
    # never hand the driver an oversized line: drop the optional parts, least important first
    for victim in ("detail", "configs_summary", "prefill_compare"):
        if len(json.dumps(out)) < HEADLINE_MAX_BYTES:
            break
        out.pop(victim, None)
    return out


# --------------------------------------------------------------------------------------------------
# the oracle arm (cpu_baseline and --impl reference)
# --------------------------------------------------------------------------------------------------
def oracle_sample(cfg, wl, seed, lib_segments, layers=1, kv_heads=None):
    """Time the CPU oracle, as it stands, on a bounded sample of task 0 of the workload: `layers` layer(s),
    the first `kv_heads` kv heads (and their q heads), all stitched tokens, all patch tokens.
    `lib_segments(s)` returns the (K, V) tensors of library segment s.
    Returns (seconds, algorithmic bytes of the sample, description)."""
    from oracle import fcg_oracle as O
    hk = kv_heads or cfg.n_kv_heads
    G = cfg.n_q_heads // cfg.n_kv_heads
    sub = synth.scaled(cfg, n_layers=layers, n_kv_heads=hk, n_q_heads=hk * G)
    task = wl.tasks[0]
    orc = O.OracleLibrary(layers, hk * G, hk, cfg.head_dim, page_size=cfg.page_size, rope_base=cfg.rope_base)
    used = sorted({s for (s, _, _, _) in task.entries})
    ids = {}
    for s in used:
        k, v = lib_segments(s)
        ids[s] = orc.segment_register(synth.to_bits(k[:layers, :hk]), synth.to_bits(v[:layers, :hk]), int(wl.orig_starts[s]))
    q, k, v = synth.patch_qkv(sub, task.task_id, len(task.positions), seed, "cpu")
    qb, kb, vb = synth.to_bits(q), synth.to_bits(k), synth.to_bits(v)
    plan = O.Plan(0, [O.PlanEntry(ids[s], b, n, d) for (s, b, n, d) in task.entries], [O.Hole(*h) for h in task.holes], task.capacity)
    t0 = time.perf_counter()
    orc.stitch([plan])
    t1 = time.perf_counter()
    orc.patch(0, 0, qb, kb, vb, task.positions)
    t2 = time.perf_counter()
    n_st = sum(n for (_, _, n, _) in task.entries)
    sb = n_st * sub.kv_bytes_per_token * 2
    ab = layers * (int(task.positions[-1]) + 1) * hk * cfg.head_dim * 4
    desc = (f"task 0 of {cfg.name}, {layers} of {cfg.n_layers} layer(s) x {hk} of {cfg.n_kv_heads} kv heads: stitch {n_st} tokens "
            f"({t1 - t0:.2f} s) + patch attention of {len(task.positions)} tokens ({t2 - t1:.2f} s)")
    return t2 - t0, sb + ab, desc


def blas_threads() -> int:
    try:
        from threadpoolctl import threadpool_info
        return max([i.get("num_threads", 1) for i in threadpool_info()] + [1])
    except Exception:
        return 1


def sample_shape(cfg, wl, seed, lib_segments, budget_s):
    """(layers, kv_heads) of a sample the oracle finishes in about `budget_s` seconds (probe: 1 layer x 2 heads)."""
    probe_heads = min(2, cfg.n_kv_heads)
    secs, _, _ = oracle_sample(cfg, wl, seed, lib_segments, 1, probe_heads)
    units = max(1.0, budget_s / (secs / probe_heads))          # (layer, kv head) units that fit
    if units >= cfg.n_kv_heads:
        return int(min(cfg.n_layers, units // cfg.n_kv_heads)), cfg.n_kv_heads
    return 1, int(units)


def cpu_baseline(cfg, wl, seed, lib_segments, budget_s=15.0):
    layers, heads = sample_shape(cfg, wl, seed, lib_segments, budget_s)
    secs, nbytes, desc = oracle_sample(cfg, wl, seed, lib_segments, layers, heads)
    return {"value": nbytes / secs / 1e9, "unit": UNIT, "cores": blas_threads(),
            "host_cpus": os.cpu_count(), "kind": "oracle", "seconds": secs,
            "sample": desc + "; numpy fp64 (elementwise single-threaded, BLAS matvec multi-threaded)"}


def run_reference(args):
    """--impl reference: the oracle IS the reference for this paper.  Rank 0 only.  Each of the K steps is the
    same bounded sample of the headline workload, sized so that warmup + K steps take about two minutes."""
    if int(os.environ.get("RANK", "0")) != 0:
        return None
    name = args.config if args.config != "all" else HEADLINE
    cfg = BENCH_CONFIGS[name]
    wl = synth.make_workload(cfg, args.seed)
    seed = args.seed
    cache = {}

    def segs(s):
        if s not in cache:
            cache[s] = synth.segment_kv(cfg, s, int(wl.seg_lens[s]), seed, "cpu")
        return cache[s]

    budget = 120.0 / (args.steps + args.warmup)
    layers, heads = sample_shape(cfg, wl, seed, segs, budget)
    times, nbytes, desc = [], 0, ""
    for i in range(args.warmup + args.steps):
        secs, nbytes, desc = oracle_sample(cfg, wl, seed, segs, layers, heads)
        if i >= args.warmup:
            times.append(secs)
    ms = float(np.mean(times)) * 1e3
    val = nbytes / (ms * 1e-3) / 1e9
    cb = {"value": val, "unit": UNIT, "cores": blas_threads(), "host_cpus": os.cpu_count(),
          "kind": "oracle", "sample": "each step = " + desc}
    return {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT,
            "n_gpus": int(os.environ.get("WORLD_SIZE", "1")), "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{cfg.name} ({name}); CPU oracle, each step = {layers} layer(s) x {heads} kv head(s) of task 0"},
            "cpu_baseline": cb, "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}


def spawn_ranks(args) -> int:
    """`python bench.py --gpus N` outside torchrun: start N ranks (one per GPU) through torch.distributed.run and pass
    the child's output through.  Rank 0 prints the JSON line."""
    import socket
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="all", choices=["all"] + sorted(BENCH_CONFIGS),
                    help="all (default): headline C4 plus C2, C3, C5 and C1 in the `configs` key; or one configuration only")
    ap.add_argument("--seed", type=int, default=1, help="layout seed of the headline numbers")
    ap.add_argument("--seeds", default="1,2,3", help="layout seeds reported per configuration (the paper's seeds)")
    ap.add_argument("--no-seeds", action="store_true", help="skip the other layout seeds")
    ap.add_argument("--page-size", type=int, default=0, choices=[0, 8, 16, 32, 64],
                    help="override the config's page size (secondary measurement; default: the config's 16)")
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--shard", default="auto", choices=["auto", "weak", "task", "head", "replica"],
                    help="multi-GPU: weak = 32 x N tasks LPT-balanced (default for the batched config), task / head = split the "
                         "single-GPU workload by task / kv head (strong scaling), replica = N identical copies")
    ap.add_argument("--devices", default="own", choices=["own", "same"],
                    help="own: rank r uses cuda:LOCAL_RANK over NCCL; same: every rank uses cuda:0 with gloo for the control plane "
                         "(exercises the multi-rank code on a 1-GPU box; the ranks' kernels never wait on one another)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-prefill-compare", action="store_true", help="skip C5's graft-vs-prefill comparison")
    ap.add_argument("--no-next", action="store_true", help="skip the NEXT-row timings (shift, extract, decode, plans)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "cuda" else args.warmup
    if args.impl == "reference":
        res = run_reference(args)
    else:
        if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
            sys.exit(spawn_ranks(args))
        res = run_cuda(args)
    if res is not None:
        if args.impl == "cuda":
            # the fat record first (own line, prefixed), the compact headline LAST: the driver parses the last stdout line
            print("DETAIL " + json.dumps(_sig(res, 7)), flush=True)
            res = headline(res)
        print(json.dumps(res, allow_nan=False), flush=True)


if __name__ == "__main__":
    main()
