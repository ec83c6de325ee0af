"""Seeded synthetic inputs for the grafting hot path.

This module serves BOTH the CUDA path's callers (tests, bench, smoke) and the
oracle's callers, so it holds none of the method's arithmetic: only shapes,
integer layout randomness and N(0,1) bf16 tensors from ``torch.Generator``.
It imports neither ``oracle`` nor the C-ABI binding.

The inputs stand in for the paper's Code-as-Policies prompts (ALFRED / TEACh /
RLBench task streams: "thousands of tokens"; FIM repair
<= 128 tokens); the benchmarks' own items are not reproduced.
Shapes follow BASELINE.json ``configs[0..4]`` (C1..C5), layout seeds 1, 2, 3
follow the paper's seeds.  Recipe: DESIGN.md "Input recipe".
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace

import numpy as np
import torch


@dataclass(frozen=True)
class GraftConfig:
    name: str
    n_layers: int
    n_q_heads: int
    n_kv_heads: int
    head_dim: int
    page_size: int
    rope_base: float
    n_segments: int
    seg_len_min: int
    seg_len_max: int
    orig_start_max: int
    n_tasks: int
    # per task: number of plan entries (min, max), composite length rule and holes
    n_entries_min: int
    n_entries_max: int
    total_tokens: int            # exact composite length T (0 -> free, see total_min/max)
    total_min: int = 0
    total_max: int = 0
    distinct_segments: bool = True
    # holes: list of (after_entry_index or -1 for "at the end", n_tokens); n_tokens <= 0 -> U{patch_min..patch_max}
    holes: tuple = ()
    patch_min: int = 0
    patch_max: int = 0

    @property
    def kv_bytes_per_token(self) -> int:
        """K and V, all layers, bf16."""
        return self.n_layers * self.n_kv_heads * self.head_dim * 2 * 2


C1 = GraftConfig("C1-tiny", 1, 8, 4, 64, 16, 1e4, 8, 64, 256, 1024, 1, 4, 4, 0,
                 holes=((1, 32),))
C2 = GraftConfig("C2-llama7b", 32, 32, 32, 128, 16, 1e4, 64, 128, 1024, 8192, 1, 6, 6, 4096,
                 holes=((2, 16), (-1, 48)))
C3 = GraftConfig("C3-llama3-8b-gqa", 32, 32, 8, 128, 16, 5e5, 64, 256, 1024, 8192, 1, 12, 12, 8192,
                 holes=((5, 64), (-1, 64)))
C4 = GraftConfig("C4-batched32", 32, 32, 8, 128, 16, 1e4, 256, 64, 1024, 8192, 32, 4, 10, 0,
                 total_min=2048, total_max=6144, distinct_segments=False,
                 holes=((-1, 0),), patch_min=8, patch_max=64)
C5 = GraftConfig("C5-long32k", 48, 64, 8, 128, 16, 1e6, 24, 1152, 1792, 32768, 1, 24, 24, 32768,
                 holes=((-1, 256),))
CONFIGS = {"C1": C1, "C2": C2, "C3": C3, "C4": C4, "C5": C5}


def scaled(cfg: GraftConfig, **kw) -> GraftConfig:
    """A copy of ``cfg`` with some fields replaced (tests shrink layer counts etc.)."""
    return replace(cfg, **kw)


@dataclass
class TaskSpec:
    task_id: int
    entries: list               # [(seg_id, src_begin, n_tokens, dst_offset)]
    holes: list                 # [(begin, n_tokens)]
    capacity: int
    positions: np.ndarray       # int32, all hole tokens in increasing order (one patch call)


@dataclass
class Workload:
    cfg: GraftConfig
    seed: int
    seg_lens: np.ndarray        # int32[n_segments]
    orig_starts: np.ndarray     # int32[n_segments]
    tasks: list = field(default_factory=list)

    @property
    def stitched_tokens(self) -> int:
        return int(sum(n for t in self.tasks for (_, _, n, _) in t.entries))

    @property
    def patch_tokens(self) -> int:
        return int(sum(len(t.positions) for t in self.tasks))


def make_workload(cfg: GraftConfig, seed: int = 1) -> Workload:
    """Integer layout of library + plans.  numpy PCG64 seeded with ``seed``."""
    rng = np.random.default_rng(seed)
    seg_lens = rng.integers(cfg.seg_len_min, cfg.seg_len_max + 1, size=cfg.n_segments).astype(np.int32)
    orig_starts = rng.integers(0, cfg.orig_start_max + 1, size=cfg.n_segments).astype(np.int32)
    wl = Workload(cfg, seed, seg_lens, orig_starts)
    for task_id in range(cfg.n_tasks):
        hole_sizes = [n if n > 0 else int(rng.integers(cfg.patch_min, cfg.patch_max + 1)) for (_, n) in cfg.holes]
        hole_total = sum(hole_sizes)
        for _attempt in range(100000):
            n_e = int(rng.integers(cfg.n_entries_min, cfg.n_entries_max + 1))
            if cfg.distinct_segments:
                ids = rng.permutation(cfg.n_segments)[:n_e]
            else:
                ids = rng.integers(0, cfg.n_segments, size=n_e)
            # sub-ranges: skip up to 1/8 of a segment's head (exercises src_begin > 0)
            begins = np.array([int(rng.integers(0, seg_lens[s] // 8 + 1)) for s in ids])
            lens = seg_lens[ids] - begins
            if cfg.total_tokens > 0:
                want = cfg.total_tokens - hole_total
                if lens[:-1].sum() < want <= lens.sum():
                    lens = lens.copy()
                    lens[-1] = want - lens[:-1].sum()          # last entry truncated by sub-range
                    break
            elif cfg.total_min > 0:
                if cfg.total_min <= lens.sum() + hole_total <= cfg.total_max:
                    break
            else:
                break
        else:
            raise RuntimeError("could not sample a plan")
        entries, holes, cursor = [], [], 0
        for idx, (s, b, n) in enumerate(zip(ids, begins, lens)):
            entries.append((int(s), int(b), int(n), cursor))
            cursor += int(n)
            for (after, _), hs in zip(cfg.holes, hole_sizes):
                if after == idx:
                    holes.append((cursor, hs))
                    cursor += hs
        for (after, _), hs in zip(cfg.holes, hole_sizes):
            if after == -1:
                holes.append((cursor, hs))
                cursor += hs
        positions = np.concatenate([np.arange(b, b + n) for (b, n) in sorted(holes)]).astype(np.int32) \
            if holes else np.zeros(0, np.int32)
        wl.tasks.append(TaskSpec(task_id, entries, holes, cursor, positions))
    return wl


# ----------------------------------------------------------------------------
# tensors
# ----------------------------------------------------------------------------
def _normal_bf16(shape, seed: int, device) -> torch.Tensor:
    g = torch.Generator(device=device)
    g.manual_seed(int(seed))
    return torch.randn(shape, generator=g, device=device, dtype=torch.float32).to(torch.bfloat16)


def segment_kv(cfg: GraftConfig, seg_idx: int, n_tokens: int, seed: int, device="cpu"):
    """K, V for one library segment: bf16 ~N(0,1), [L][Hkv][n][D]."""
    shape = (cfg.n_layers, cfg.n_kv_heads, int(n_tokens), cfg.head_dim)
    base = 1_000_003 * int(seed) + 2 * int(seg_idx)
    return _normal_bf16(shape, base, device), _normal_bf16(shape, base + 1, device)


def patch_qkv(cfg: GraftConfig, task_id: int, n: int, seed: int, device="cpu"):
    """q [L][n][Hq][D], k, v [L][n][Hkv][D]: bf16 ~N(0,1) (already position-encoded as far as the path cares)."""
    base = 7_000_003 * int(seed) + 3 * int(task_id) + 500_000_000
    q = _normal_bf16((cfg.n_layers, n, cfg.n_q_heads, cfg.head_dim), base, device)
    k = _normal_bf16((cfg.n_layers, n, cfg.n_kv_heads, cfg.head_dim), base + 1, device)
    v = _normal_bf16((cfg.n_layers, n, cfg.n_kv_heads, cfg.head_dim), base + 2, device)
    return q, k, v


def to_bits(t: torch.Tensor) -> np.ndarray:
    """bf16 tensor -> uint16 numpy array of the same shape (reinterpretation, no arithmetic)."""
    return t.detach().contiguous().cpu().view(torch.int16).numpy().view(np.uint16)


def from_bits(a: np.ndarray, device="cpu") -> torch.Tensor:
    """uint16 numpy array -> bf16 tensor (reinterpretation)."""
    return torch.from_numpy(np.ascontiguousarray(a).view(np.int16)).view(torch.bfloat16).to(device)
