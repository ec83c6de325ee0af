"""bench.py -- one "step" = one pass of the whole grafting hot path (S2 plan -> S3 fused gather +
RoPE-shift -> S4 scatter -> S5/S6 patch attention, all layers) over one synthetic batch.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C2] [--impl reference]

Prints ONE JSON line (rank 0).  metric = BASELINE.json's: graft latency (ms_per_step) and achieved
algorithmic HBM GB/s (value) against the roofline on a B200.  Multi-GPU: the path shards by task
(independent grafting tasks, no collective): every rank grafts its own copy of the workload
("scaling": "weak").  --impl reference times the CPU oracle (the only reference this paper has).
"""
from __future__ import annotations

import argparse
import json
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

from paper_2606_13097_b200 import synth  # noqa: E402

METRIC = "graft latency ms + HBM GB/s (stitch+RoPE shift, patch attn) vs roofline, 1 B200"
FALLBACK_HBM_GBS = 6650.0          # B200_PROFILING.md fallback, used only if MEASURED_PEAKS.json is absent


def peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            p = json.load(f)
        return float(p["hbm_gbs"]), "measured (MEASURED_PEAKS.json, torch copy_ read+write)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


# --------------------------------------------------------------------------------------------------
# algorithmic bytes
# --------------------------------------------------------------------------------------------------
def stitch_bytes(cfg, wl) -> int:
    """every stitched K/V byte is read once and written once: T_stitched * L * Hkv * D * 2 B * 2 (K,V) * 2 (r+w)."""
    return wl.stitched_tokens * cfg.kv_bytes_per_token * 2


def attn_bytes(cfg, wl) -> int:
    """visible K+V read once per kv head: sum over tasks of L * kv_len * Hkv * D * 4 B (q/out/partials < 1 %)."""
    total = 0
    for t in wl.tasks:
        kv_len = int(t.positions[-1]) + 1
        total += cfg.n_layers * kv_len * cfg.n_kv_heads * cfg.head_dim * 4
    return total


def attn_flops(cfg, wl) -> int:
    """Q K^T and P V over the visible cache only: per layer, q head and patch token i, 4 * D * (p_i + 1) flops."""
    vis = sum(int((np.asarray(t.positions, np.int64) + 1).sum()) for t in wl.tasks)
    return 4 * cfg.head_dim * cfg.n_layers * cfg.n_q_heads * vis


def attn_rows(cfg, wl) -> int:
    """largest R = n * G (query rows per kv head) of the batch: intensity of patch attention is R flop/B."""
    return max(len(t.positions) for t in wl.tasks) * (cfg.n_q_heads // cfg.n_kv_heads)


# dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed `ncu --set full` captures
# (profiles/r01_final.md); None where no capture of that workload is committed.
NCU_TRAFFIC = {"C2": {"stitch": 4.178e9, "attn": 2.183e9}, "C3": {"stitch": 2.061e9, "attn": 1.137e9},
               "C4": {"stitch": 30.15e9, "attn": 16.14e9}, "C5": {"attn": 6.993e9}}


def tensor_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            p = json.load(f)
        return float(p["bf16_tflops_sustained"]), "measured (MEASURED_PEAKS.json, sustained bf16 matmul)"
    except Exception:
        return 1400.0, "fallback (B200_PROFILING.md, sustained)"


EXTRACT_TOKENS = 1024


def time_next_rows(lib, cfg, wl, seed, dev, iters=5):
    """SURVEY.md 8(f) NEXT rows, timed on task 0 of the stitched workload after the main measurement (CUDA events,
    2 warm-ups): suffix re-graft by -16 / +16 tokens (fcg_task_shift), extraction of EXTRACT_TOKENS tokens into the
    library (fcg_segment_extract), and one decode step (fcg_patch, n = 1, R = G) over the whole cache."""
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

    res = {}
    # the call pattern of a model that patches layer by layer: L calls of one layer each (task 0's own patch tokens)
    try:
        qp, kp, vp = synth.patch_qkv(cfg, t.task_id, len(t.positions), seed, dev)
        op = torch.empty_like(qp)
        views = [(qp[l:l + 1], kp[l:l + 1], vp[l:l + 1], op[l:l + 1]) for l in range(cfg.n_layers)]

        def per_layer():
            for l, (a_, b_, c_, d_) in enumerate(views):
                lib.patch(t.task_id, l, a_, b_, c_, t.positions, d_)

        for _ in range(2):
            per_layer()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize(dev)
        t0 = time.perf_counter()
        a.record()
        for _ in range(iters):
            per_layer()
        b.record()
        t1 = time.perf_counter()
        torch.cuda.synchronize(dev)
        res["patch_one_call_per_layer"] = {"ms": a.elapsed_time(b) / iters, "host_enqueue_ms": (t1 - t0) * 1e3 / iters,
                                           "calls": cfg.n_layers, "splits": lib.stats()["last_attn_splits"],
                                           "note": "same patch as the timed step, issued as one fcg_patch per layer"}
        del qp, kp, vp, op, views
    except Exception as e:
        res["patch_one_call_per_layer"] = {"error": repr(e)}
    per_tok = cfg.kv_bytes_per_token
    for name, fn, nbytes in (("decode_step", decode, cfg.n_layers * cap * cfg.n_kv_heads * cfg.head_dim * 4),
                             ("segment_register", register, n_ext * per_tok * 2),
                             ("segment_extract", extract, n_ext * per_tok * 2),
                             ("task_shift", shift_pair, 2 * n_shift * per_tok * 2)):
        for _ in range(2):
            fn()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize(dev)
        a.record()
        for _ in range(iters):
            fn()
        b.record()
        torch.cuda.synchronize(dev)
        ms = a.elapsed_time(b) / iters
        res[name] = {"ms": ms, "GBps": nbytes / (ms * 1e-3) / 1e9, "bytes": int(nbytes)}
    # NEXT-3 two-tier residency: one library segment to the pinned host tier and back (copy engine), and a stitch
    # that reads it in place from the host tier (zero-copy over the host link)
    seg = int(t.entries[0][0])
    n_seg = int(wl.seg_lens[seg])
    seg_bytes = n_seg * per_tok
    try:
        lib.task_release(t.task_id)
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
        host_ms = timed(lambda: lib.stitch(plan), before=lambda: lib.pool_info()["n_tasks_live"] and lib.task_release(t.task_id))
        lib.task_release(t.task_id)
        lib.segment_prefetch(seg)
        res["segment_offload"] = {"ms": off_ms, "GBps": seg_bytes / (off_ms * 1e-3) / 1e9, "bytes": int(seg_bytes)}
        res["segment_prefetch"] = {"ms": pre_ms, "GBps": seg_bytes / (pre_ms * 1e-3) / 1e9, "bytes": int(seg_bytes)}
        res["stitch_from_host_tier"] = {"ms": host_ms, "GBps": seg_bytes / (host_ms * 1e-3) / 1e9, "bytes": int(seg_bytes),
                                        "note": f"{n_seg}-token segment read in place from pinned host memory (bytes = one-way)"}
    except Exception as e:
        res["two_tier"] = {"error": repr(e)}
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
    except Exception as e:
        res["torch_sdpa_ms_all_layers"] = None
        res["torch_sdpa_error"] = repr(e)
    lib.task_release(t.task_id)
    return res


class ClockSampler:
    """nvidia-smi clocks + throttle reasons during the timed region (B200_PROFILING.md recipe).  nvidia-smi is started
    before the warm-up (it needs ~0.1 s to come up) and samples every 20 ms; rows are time-stamped on arrival and
    only those inside [mark_begin, mark_end] count.  If the region was too short to catch one, the rows nearest to
    it (within 0.3 s, i.e. warm-up steps of the same workload) are used and `window` says so."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None
        self.t0 = self.t1 = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "20", "-i", str(self.index)], stdout=subprocess.PIPE, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), [x.strip() for x in line.split(",")]))

    def mark_begin(self):
        self.t0 = time.time()

    def mark_end(self):
        self.t1 = time.time()

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.05)
        self.proc.terminate()
        t0, t1 = self.t0 or 0.0, self.t1 or time.time()
        inside = [r for (ts, r) in self.rows if t0 <= ts <= t1 + 0.02]
        window = "timed region"
        if not inside:
            inside = [r for (ts, r) in self.rows if t0 - 0.3 <= ts <= t1 + 0.3]
            window = "nearest samples within 0.3 s of the timed region (region shorter than the sampling period)"
        sm, smax, reasons = [], [], set()
        for r in inside:
            try:
                sm.append(float(r[1])), smax.append(float(r[2]))
            except Exception:
                continue
            for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[5:9]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "reasons": sorted(reasons), "samples": len(sm), "window": window}


# --------------------------------------------------------------------------------------------------
# the CUDA arm
# --------------------------------------------------------------------------------------------------
def build_library(cfg, wl, seed, device_index, on_segment=None):
    """The library exactly as the timed run uses it.  `on_segment(s, k, v)` lets the full-size parity tests
    keep slices of the device-generated segments for the oracle."""
    from paper_2606_13097_b200 import binding
    total_pages = sum(-(-t.capacity // cfg.page_size) for t in wl.tasks)
    # + EXTRACT_TOKENS of arena and + half a task of pages: room for the NEXT-row measurements (segment extraction,
    # copy-on-shift); neither changes what the graft step itself touches
    seg_tokens = int(wl.seg_lens.sum()) + EXTRACT_TOKENS
    total_pages += max(-(-t.capacity // cfg.page_size) for t in wl.tasks) // 2 + 8
    lib = binding.FcgLibrary(n_layers=cfg.n_layers, n_q_heads=cfg.n_q_heads, n_kv_heads=cfg.n_kv_heads,
                             head_dim=cfg.head_dim, page_size=cfg.page_size, rope_base=cfg.rope_base,
                             max_segments=cfg.n_segments + 1, max_tasks=max(cfg.n_tasks, 1),
                             max_task_tokens=max(t.capacity for t in wl.tasks), n_pages=total_pages + 16,
                             workspace_bytes=2 << 30, segment_tokens=seg_tokens, device=device_index,
                             host_tier_tokens=int(wl.seg_lens[wl.tasks[0].entries[0][0]]) + 16)
    dev = torch.device("cuda", device_index)
    for s in range(cfg.n_segments):
        k, v = synth.segment_kv(cfg, s, int(wl.seg_lens[s]), seed, dev)
        sid = lib.segment_register(k, v, int(wl.orig_starts[s]))
        assert sid == s
        if on_segment is not None:
            on_segment(s, k, v)
        del k, v
    torch.cuda.synchronize(dev)
    return lib


def plans_for(wl):
    return [{"task_id": t.task_id, "entries": t.entries, "holes": t.holes, "capacity_tokens": t.capacity} for t in wl.tasks]


def run_cuda(args, cfg, wl, seed):
    from paper_2606_13097_b200 import binding
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    lib = build_library(cfg, wl, seed, local)
    plans = plans_for(wl)
    ids = [t.task_id for t in wl.tasks]
    npt = [len(t.positions) for t in wl.tasks]
    pos = np.concatenate([t.positions for t in wl.tasks]).astype(np.int32)
    n_total = int(pos.size)
    qs = [synth.patch_qkv(cfg, t.task_id, len(t.positions), seed, dev) for t in wl.tasks]
    q = torch.cat([x[0] for x in qs], dim=1).contiguous()
    k = torch.cat([x[1] for x in qs], dim=1).contiguous()
    v = torch.cat([x[2] for x in qs], dim=1).contiguous()
    out = torch.empty_like(q)
    del qs
    live = [False]

    def step_device(ev=None):
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

    def barrier():
        torch.cuda.synchronize(dev)
        if world > 1:
            import torch.distributed as dist
            dist.barrier()
        torch.cuda.synchronize(dev)

    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    for _ in range(args.warmup):
        step_device()
    barrier()
    s0 = lib.stats()
    sampler.mark_begin()
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(args.steps)]
    t_begin, t_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t_begin.record()
    for i in range(args.steps):
        step_device(evs[i])
    t_end.record()
    barrier()
    sampler.mark_end()
    clocks = sampler.stop() if rank == 0 else None
    s1 = lib.stats()
    total_ms = t_begin.elapsed_time(t_end)
    stitch_ms = [e[0].elapsed_time(e[1]) for e in evs]
    patch_ms = [e[1].elapsed_time(e[2]) for e in evs]
    if world > 1:
        import torch.distributed as dist
        tt = torch.tensor([total_ms], device=dev)
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        total_ms = float(tt.item())
    ms_per_step = total_ms / args.steps
    launches = sum(s1[f] - s0[f] for f in s1 if f.endswith("_launches"))

    # ---- e2e: same step through the C ABI with HOST buffers (H2D of q/k/v, D2H of out inside) ----
    single = len(ids) == 1
    e2e = None
    if True:
        qh, kh, vh = [x.cpu().contiguous().pin_memory() for x in (q, k, v)]
        oh = torch.empty_like(qh).pin_memory()

        def step_host():
            for tid in ids:
                lib.task_release(tid)
            lib.stitch(plans)
            if single:
                lib.patch_host(ids[0], 0, qh, kh, vh, pos, oh)
            else:
                lib.patch_batch_host(ids, npt, 0, qh, kh, vh, pos, oh)
            torch.cuda.synchronize(dev)          # the caller reads `out` on the host every step

        for _ in range(min(args.warmup, 3)):
            step_host()
        barrier()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(args.steps):
            step_host()
        b.record()
        barrier()
        e2e_ms = a.elapsed_time(b) / args.steps
        if world > 1:
            import torch.distributed as dist
            tt = torch.tensor([e2e_ms], device=dev)
            dist.all_reduce(tt, op=dist.ReduceOp.MAX)
            e2e_ms = float(tt.item())
        h2d = int(qh.numel() + kh.numel() + vh.numel()) * 2
        d2h = int(oh.numel()) * 2
        e2e = (e2e_ms, h2d, d2h)
        assert torch.equal(oh, out.cpu()), "host-buffer call and device call disagree"

    sb, ab = stitch_bytes(cfg, wl), attn_bytes(cfg, wl)
    peak, peak_src = peaks()
    # patch attention: HBM-bound while R = n*G (flop per byte) is small, tensor-bound from R ~ 250
    af, rows = attn_flops(cfg, wl), attn_rows(cfg, wl)
    attn_s = float(np.mean(patch_ms)) * 1e-3
    if rows >= 250:
        tpeak, tsrc = tensor_peak()
        attn_roof = {"bound": "tensor", "achieved": af / attn_s / 1e12, "peak": tpeak, "unit": "TFLOP/s",
                     "frac": af / attn_s / 1e12 / tpeak, "peak_source": tsrc, "rows_per_kv_head": rows,
                     "hbm_GBps": ab / attn_s / 1e9}
    else:
        attn_roof = {"bound": "hbm", "achieved": ab / attn_s / 1e9, "peak": peak, "unit": "GB/s",
                     "frac": ab / attn_s / 1e9 / peak, "frac_of_8TBps": ab / attn_s / 1e9 / 8000.0,
                     "rows_per_kv_head": rows, "TFLOPs": af / attn_s / 1e12}
    attn_roof["traffic"] = NCU_TRAFFIC.get(args.config, {}).get("attn")
    attn_roof["note"] = "timed as scatter + attention (+ combine); scatter is ~1 % of it"
    res = {
        "metric": METRIC, "value": world * (sb + ab) / (ms_per_step * 1e-3) / 1e9, "unit": "GB/s (algorithmic, whole graft)",
        "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_per_step,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
        "config": {"workload": f"{cfg.name} ({args.config}): L={cfg.n_layers} Hq={cfg.n_q_heads} Hkv={cfg.n_kv_heads} "
                               f"D={cfg.head_dim} page={cfg.page_size} base={cfg.rope_base:g}; library {cfg.n_segments} segments "
                               f"({int(wl.seg_lens.sum())} tokens); {len(wl.tasks)} task(s), {wl.stitched_tokens} stitched + "
                               f"{wl.patch_tokens} patch tokens; layout seed {seed}",
                   "l2": "inputs larger than L2 (each step streams >= 1 GiB; no flush needed)" if sb > 4 * 126e6
                   else "working set fits L2: latency only, no roofline claim",
                   "stitch_ms": float(np.mean(stitch_ms)), "stitch_ms_min": float(np.min(stitch_ms)),
                   "stitch_ms_median": float(np.median(stitch_ms)),
                   "patch_ms": float(np.mean(patch_ms)), "patch_ms_min": float(np.min(patch_ms)),
                   "patch_ms_median": float(np.median(patch_ms)),
                   "stitch_GBps": sb / (np.mean(stitch_ms) * 1e-3) / 1e9, "patch_attn_GBps": ab / (np.mean(patch_ms) * 1e-3) / 1e9,
                   "stitch_bytes": sb, "attn_bytes": ab, "attn_path": s1["last_attn_path"], "attn_splits": s1["last_attn_splits"],
                   "parallelism": f"task-replica x{world}"},
        "gpu_launches": int(launches),
        "roofline": {"kernel": "stitch_kernel (fused gather + RoPE-shift)", "bound": "hbm",
                     "achieved": sb / (np.mean(stitch_ms) * 1e-3) / 1e9, "peak": peak, "unit": "GB/s",
                     "frac": sb / (np.mean(stitch_ms) * 1e-3) / 1e9 / peak, "peak_source": peak_src,
                     "frac_of_8TBps": sb / (np.mean(stitch_ms) * 1e-3) / 1e9 / 8000.0,
                     "traffic": args.traffic if args.traffic is not None else NCU_TRAFFIC.get(args.config, {}).get("stitch"),
                     "patch_attention": attn_roof},
        "clocks": clocks,
    }
    if e2e:
        res["e2e"] = {"value": world * (sb + ab) / (e2e[0] * 1e-3) / 1e9, "unit": "GB/s (algorithmic, whole graft)",
                      "ms_per_step": e2e[0], "h2d_bytes_per_step": e2e[1], "d2h_bytes_per_step": e2e[2]}
    if rank == 0 and not args.no_next:
        try:
            res["next_rows"] = time_next_rows(lib, cfg, wl, seed, dev)
        except Exception as e:       # never lose the main line to an extra
            res["next_rows"] = {"error": repr(e)}
    if rank == 0 and args.prefill_compare:
        try:
            res["prefill_compare"] = time_prefill_compare(lib, cfg, wl, seed, dev)
            res["prefill_compare"]["graft_ms"] = ms_per_step
            res["prefill_compare"]["prefill_attention_over_graft"] = res["prefill_compare"]["own_kernel_ms_all_layers"] / ms_per_step
        except Exception as e:
            res["prefill_compare"] = {"error": repr(e)}
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        res["cpu_baseline"] = cpu_baseline(cfg, wl, seed, lib_segments=lambda s: synth.segment_kv(cfg, s, int(wl.seg_lens[s]), seed, dev))
    lib.close()
    if world > 1:
        import torch.distributed as dist
        dist.barrier()                      # rank 0 may still have been timing its extras
        dist.destroy_process_group()
    return res if rank == 0 else None


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
    return {"value": nbytes / secs / 1e9, "unit": "GB/s (algorithmic, whole graft)", "cores": blas_threads(),
            "host_cpus": os.cpu_count(), "kind": "oracle", "seconds": secs,
            "sample": desc + "; numpy fp64 (elementwise single-threaded, BLAS matvec multi-threaded)"}


def run_reference(args, cfg, wl, seed):
    """--impl reference: the oracle IS the reference for this paper.  Rank 0 only.  Each of the K steps is the
    same bounded sample, sized so that warmup + K steps take about two minutes."""
    if int(os.environ.get("RANK", "0")) != 0:
        return None
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
    unit = "GB/s (algorithmic, whole graft)"
    cb = {"value": val, "unit": unit, "cores": blas_threads(), "host_cpus": os.cpu_count(),
          "kind": "oracle", "sample": "each step = " + desc}
    return {"impl": "reference", "metric": METRIC, "value": val, "unit": unit,
            "n_gpus": int(os.environ.get("WORLD_SIZE", "1")), "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{cfg.name} ({args.config}); CPU oracle, each step = {layers} layer(s) x {heads} kv head(s) of task 0"},
            "cpu_baseline": cb, "e2e": {"value": val, "unit": unit, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="C2", choices=sorted(synth.CONFIGS))
    ap.add_argument("--seed", type=int, default=1)
    ap.add_argument("--page-size", type=int, default=0, choices=[0, 8, 16, 32, 64],
                    help="override the config's page size (secondary measurement; default: the config's 16)")
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--prefill-compare", action="store_true",
                    help="also time causal prefill attention over the task's whole length (C5's comparison)")
    ap.add_argument("--no-next", action="store_true", help="skip the NEXT-row timings (shift, extract, decode)")
    ap.add_argument("--traffic", type=float, default=None, help="ncu dram bytes per stitch launch, if known (profiles/)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "cuda" else args.warmup
    cfg = synth.CONFIGS[args.config]
    if args.page_size:
        cfg = synth.scaled(cfg, page_size=args.page_size)
    wl = synth.make_workload(cfg, args.seed)
    if args.impl == "reference":
        res = run_reference(args, cfg, wl, args.seed)
    else:
        res = run_cuda(args, cfg, wl, args.seed)
    if res is not None:
        print(json.dumps(res))


if __name__ == "__main__":
    main()
