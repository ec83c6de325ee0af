"""Shared test plumbing: drive the oracle and the CUDA library from the same seeded workload and
compare.  Holds no arithmetic of the method (comparisons only)."""
from __future__ import annotations

import numpy as np
import torch

from oracle import fcg_oracle as O
from paper_2606_13097_b200 import synth

ATTN_RTOL, ATTN_ATOL = 2e-2, 1e-2      # north_star: "within 2e-2 relative and 1e-2 absolute"


def ulp_key(bits: np.ndarray) -> np.ndarray:
    """monotone integer image of bf16 bit patterns (sign-magnitude -> two's complement order)."""
    b = bits.astype(np.int32)
    return np.where(b & 0x8000, -(b & 0x7FFF), b)


def ulp_dist(a_bits: np.ndarray, b_bits: np.ndarray) -> np.ndarray:
    return np.abs(ulp_key(np.asarray(a_bits)) - ulp_key(np.asarray(b_bits)))


def assert_k_within_1ulp(gpu_bits, ref_bits, what=""):
    d = ulp_dist(gpu_bits, ref_bits)
    hist = np.bincount(np.minimum(d.ravel(), 3), minlength=4)
    assert hist[2] + hist[3] == 0, f"{what}: shifted K ulp histogram [0,1,2,>=3] = {hist.tolist()}"
    return hist


def k_pair_close(a_bits, b_bits, c, rope_mode=1):
    """|a - b| <= c * 2^-9 * |rotation pair| per component: the bar for keys that went through MORE than one rotation
    generation (each side rounds once per generation, from inputs that may already differ by a rounding), where a ulp
    count is meaningless for the small component of a pair."""
    a, b = O.bf16_to_f64(np.asarray(a_bits)), O.bf16_to_f64(np.asarray(b_bits))
    if rope_mode == 2:
        norm = np.repeat(np.sqrt(b[..., 0::2] ** 2 + b[..., 1::2] ** 2), 2, axis=-1)
    else:
        half = b.shape[-1] // 2
        n = np.sqrt(b[..., :half] ** 2 + b[..., half:] ** 2)
        norm = np.concatenate([n, n], axis=-1)
    return bool(np.all(np.abs(a - b) <= c * 2.0 ** -9 * norm + 1e-30))


# Regression guard for the FULL-SIZE attention tests, beside north_star's tolerance (which stays the acceptance bar): with
# N(0,1) inputs and thousands of visible tokens the outputs are ~0.01-0.03, so atol = 1e-2 alone cannot see a dropped
# 64-token tile.  Per (layer, kv head, task) slice: rms(gpu - oracle) <= RMS_GUARD * rms(oracle).  bf16 rounding of P and
# of the output gives 0.2-0.4 %; tests/test_attention_guard.py shows which faults exceed the guard at C2's and C5's shapes.
RMS_GUARD = 0.01


def rel_rms(got: np.ndarray, ref: np.ndarray) -> float:
    return float(np.sqrt(np.mean((got - ref) ** 2)) / max(np.sqrt(np.mean(ref ** 2)), 1e-300))


def assert_attn_close(gpu_out: torch.Tensor, ref: np.ndarray, what="", rms_guard=False):
    got = gpu_out.detach().float().cpu().numpy().astype(np.float64)
    err = np.abs(got - ref)
    tol = ATTN_ATOL + ATTN_RTOL * np.abs(ref)
    bad = err > tol
    assert not bad.any(), (f"{what}: {int(bad.sum())} of {bad.size} attention outputs out of tolerance; "
                           f"max abs err {err.max():.4g}, worst ratio {(err / tol).max():.3g}")
    if rms_guard:
        r = rel_rms(got, ref)
        assert r <= RMS_GUARD, f"{what}: rms error is {100 * r:.3g} % of the output's rms (regression guard {100 * RMS_GUARD:g} %)"
    return float(err.max())


def plans_of(wl: synth.Workload, seg_ids):
    """C-ABI style plan dicts and oracle Plan objects for every task of a workload."""
    c_plans, o_plans = [], []
    for t in wl.tasks:
        ents = [(seg_ids[s], b, n, d) for (s, b, n, d) in t.entries]
        c_plans.append({"task_id": t.task_id, "entries": ents, "holes": list(t.holes), "capacity_tokens": t.capacity})
        o_plans.append(O.Plan(t.task_id, [O.PlanEntry(*e) for e in ents], [O.Hole(*h) for h in t.holes], t.capacity))
    return c_plans, o_plans


def make_pair(cfg: synth.GraftConfig, wl: synth.Workload, seed: int, *, n_pages=None, max_tasks=None,
              workspace_bytes=0, only_segments=None, rope_mode=1, inv_freq=None, host_tier_tokens=0, max_task_tokens=None):
    """Create oracle + CUDA library holding the same segment bits.  Returns (orc, lib, seg_ids)."""
    from paper_2606_13097_b200.binding import FcgLibrary
    used = sorted({s for t in wl.tasks for (s, _, _, _) in t.entries}) if only_segments is None else only_segments
    cap_tokens = max_task_tokens or max(t.capacity for t in wl.tasks)
    total_pages = sum(-(-t.capacity // cfg.page_size) for t in wl.tasks)
    n_pages = n_pages or total_pages + 8
    seg_tokens = int(sum(int(wl.seg_lens[s]) for s in used))
    lib = FcgLibrary(n_layers=cfg.n_layers, n_q_heads=cfg.n_q_heads, n_kv_heads=cfg.n_kv_heads, head_dim=cfg.head_dim,
                     page_size=cfg.page_size, rope_mode=rope_mode, rope_base=cfg.rope_base, inv_freq=inv_freq,
                     max_segments=max(len(used), 1), max_tasks=max_tasks or max(len(wl.tasks), 1),
                     max_task_tokens=cap_tokens, n_pages=n_pages, workspace_bytes=workspace_bytes,
                     segment_tokens=seg_tokens, host_tier_tokens=host_tier_tokens)
    orc = O.OracleLibrary(cfg.n_layers, cfg.n_q_heads, cfg.n_kv_heads, cfg.head_dim, page_size=cfg.page_size,
                          rope_mode=rope_mode, rope_base=cfg.rope_base, inv_freq=inv_freq,
                          max_segments=max(len(used), 1), max_tasks=max_tasks or max(len(wl.tasks), 1), n_pages=n_pages,
                          max_task_tokens=cap_tokens)
    seg_ids = {}
    for s in used:
        k, v = synth.segment_kv(cfg, s, int(wl.seg_lens[s]), seed, "cpu")
        sid_o = orc.segment_register(synth.to_bits(k), synth.to_bits(v), int(wl.orig_starts[s]))
        sid_g = lib.segment_register(k.cuda(), v.cuda(), int(wl.orig_starts[s]))
        assert sid_o == sid_g
        seg_ids[s] = sid_g
    torch.cuda.synchronize()
    return orc, lib, seg_ids


def compare_stitched(orc, lib, wl, check_all_layers=True):
    """page tables bit-exact, V bit-exact, K within 1 ulp, over the FILLED positions of every task."""
    hist_total = np.zeros(4, np.int64)
    for t in wl.tasks:
        ot = orc.tasks[t.task_id]
        assert np.array_equal(lib.task_page_table_host(t.task_id), np.asarray(ot.page_table, np.int32))
        dev_ptr, n_pages, n_tokens = lib.task_page_table(t.task_id)
        assert n_pages == len(ot.page_table) and n_tokens == ot.n_tokens
        filled = ot.filled
        layers = range(orc.L) if check_all_layers else (0, orc.L - 1)
        for layer in layers:
            k, v = lib.task_read(t.task_id, layer, 0, ot.capacity)
            kb, vb = synth.to_bits(k), synth.to_bits(v)
            assert np.array_equal(vb[:, filled], ot.v[layer][:, filled]), f"V gather not bit-exact (task {t.task_id} layer {layer})"
            hist_total += assert_k_within_1ulp(kb[:, filled], ot.k[layer][:, filled], f"task {t.task_id} layer {layer}")
    return hist_total


def run_patch_both(orc, lib, cfg, task: synth.TaskSpec, seed, positions=None, layer_begin=0, n_layers=None):
    positions = task.positions if positions is None else np.asarray(positions, np.int32)
    n_layers = n_layers or cfg.n_layers
    q, k, v = synth.patch_qkv(cfg, task.task_id, len(positions), seed, "cpu")
    q, k, v = q[layer_begin:layer_begin + n_layers], k[layer_begin:layer_begin + n_layers], v[layer_begin:layer_begin + n_layers]
    ref = orc.patch(task.task_id, layer_begin, synth.to_bits(q), synth.to_bits(k), synth.to_bits(v), positions)
    out = lib.patch(task.task_id, layer_begin, q.cuda().contiguous(), k.cuda().contiguous(), v.cuda().contiguous(), positions)
    torch.cuda.synchronize()
    return out, ref


def compare_cache_bits(orc, lib, task_id, positions):
    """after a patch: the scattered K/V rows are bit-exact in every layer."""
    ot = orc.tasks[task_id]
    for layer in range(orc.L):
        k, v = lib.task_read(task_id, layer, 0, ot.capacity)
        kb, vb = synth.to_bits(k), synth.to_bits(v)
        assert np.array_equal(kb[:, positions], ot.k[layer][:, positions]), f"K scatter not bit-exact (layer {layer})"
        assert np.array_equal(vb[:, positions], ot.v[layer][:, positions]), f"V scatter not bit-exact (layer {layer})"
