"""Host-side sharding of the grafting path over ranks.

The path shards two ways and neither needs a data-path collective:

* **task-parallel** -- grafting tasks are independent (BASELINE.json configs[3]: 32 concurrent tasks over a
  shared library): ``assign_tasks`` balances them over ranks by their byte cost; every rank stitches and patches
  only its own tasks;
* **head-parallel** -- stitch, scatter and patch attention are independent per kv head: rank r holds kv heads
  ``kv_head_range(Hkv, r, N)`` of the library and of every composite cache plus the matching q heads; plans and
  page tables are replicated integers.  Outputs stay head-sharded (what a tensor-parallel o_proj consumes).

Only *results* are ever exchanged (``gather_task_outputs`` / ``gather_head_outputs``, for callers that want the
whole tensor on one rank, e.g. the tests); they use whatever ``torch.distributed`` backend the caller initialised
(NCCL on GPUs, gloo in the CPU tests).  This module holds integers and tensor slicing only -- none of the
method's arithmetic -- and imports neither the oracle nor the C-ABI binding.
"""
from __future__ import annotations

from dataclasses import replace

import numpy as np
import torch


# --------------------------------------------------------------------------------------------------
# task-parallel
# --------------------------------------------------------------------------------------------------
def task_cost(task, kv_bytes_per_token: int = 1) -> int:
    """Algorithmic bytes of one task: stitched tokens moved twice (read + write) + the visible cache read once by
    its patch.  ``task`` is a ``synth.TaskSpec``-like object."""
    stitched = sum(n for (_, _, n, _) in task.entries)
    visible = int(task.positions[-1]) + 1 if len(task.positions) else 0
    return (2 * stitched + visible) * kv_bytes_per_token


def assign_tasks(costs, world: int) -> list[list[int]]:
    """Longest-processing-time-first assignment of task indices to ranks.  Deterministic: ties go to the lower
    task index, then the lower rank.  Returns, per rank, its task indices in ascending order."""
    if world <= 0:
        raise ValueError("world must be > 0")
    order = sorted(range(len(costs)), key=lambda i: (-int(costs[i]), i))
    load = [0] * world
    mine: list[list[int]] = [[] for _ in range(world)]
    for i in order:
        r = min(range(world), key=lambda x: (load[x], x))
        mine[r].append(i)
        load[r] += int(costs[i])
    return [sorted(m) for m in mine]


def token_slices(n_per_task) -> list[slice]:
    """Row range of every task inside the concatenated q/k/v/out/positions arrays."""
    off, out = 0, []
    for n in n_per_task:
        out.append(slice(off, off + int(n)))
        off += int(n)
    return out


def gather_task_outputs(local_out: torch.Tensor, my_tasks, n_per_task, assignment, group=None) -> torch.Tensor:
    """Reassemble ``[L][n_total][Hq][D]`` in the original task order on every rank.

    ``local_out`` holds this rank's tasks (``my_tasks``, ascending) concatenated along dim 1.  One all_gather of
    padded buffers; a result exchange, not part of the grafting path."""
    import torch.distributed as dist
    world = dist.get_world_size(group)
    sl = token_slices(n_per_task)
    rows = [sum(int(n_per_task[i]) for i in a) for a in assignment]
    pad = max(rows + [1])
    L, _, H, D = local_out.shape
    buf = local_out.new_zeros((L, pad, H, D))
    buf[:, : local_out.shape[1]] = local_out
    bufs = [torch.empty_like(buf) for _ in range(world)]
    dist.all_gather(bufs, buf, group=group)
    full = local_out.new_empty((L, sum(int(n) for n in n_per_task), H, D))
    for r, a in enumerate(assignment):
        off = 0
        for i in a:
            n = int(n_per_task[i])
            full[:, sl[i]] = bufs[r][:, off:off + n]
            off += n
    return full


# --------------------------------------------------------------------------------------------------
# head-parallel
# --------------------------------------------------------------------------------------------------
def kv_head_range(n_kv_heads: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous kv heads of ``rank``; requires ``world`` to divide ``n_kv_heads`` (equal shards, so that every
    rank launches the same grid)."""
    if n_kv_heads % world:
        raise ValueError(f"world size {world} does not divide n_kv_heads {n_kv_heads}")
    per = n_kv_heads // world
    return rank * per, (rank + 1) * per


def q_head_range(n_q_heads: int, n_kv_heads: int, rank: int, world: int) -> tuple[int, int]:
    g = n_q_heads // n_kv_heads
    b, e = kv_head_range(n_kv_heads, rank, world)
    return b * g, e * g


def head_sharded_config(cfg, rank: int, world: int):
    """The ``synth.GraftConfig`` one rank creates its library with (fewer heads, everything else equal)."""
    b, e = kv_head_range(cfg.n_kv_heads, rank, world)
    g = cfg.n_q_heads // cfg.n_kv_heads
    return replace(cfg, n_kv_heads=e - b, n_q_heads=(e - b) * g)


def slice_kv_heads(x: torch.Tensor, n_kv_heads: int, rank: int, world: int, dim: int) -> torch.Tensor:
    """This rank's kv heads of a segment tensor ``[L][Hkv][n][D]`` (dim=1) or patch k/v ``[L][n][Hkv][D]`` (dim=2)."""
    b, e = kv_head_range(n_kv_heads, rank, world)
    return x.narrow(dim, b, e - b).contiguous()


def slice_q_heads(q: torch.Tensor, n_q_heads: int, n_kv_heads: int, rank: int, world: int) -> torch.Tensor:
    b, e = q_head_range(n_q_heads, n_kv_heads, rank, world)
    return q.narrow(2, b, e - b).contiguous()


def gather_head_outputs(local_out: torch.Tensor, group=None) -> torch.Tensor:
    """Concatenate head-sharded outputs ``[L][n][Hq/N][D]`` along the head axis (rank order) on every rank."""
    import torch.distributed as dist
    world = dist.get_world_size(group)
    bufs = [torch.empty_like(local_out) for _ in range(world)]
    dist.all_gather(bufs, local_out.contiguous(), group=group)
    return torch.cat(bufs, dim=2)


def max_over_ranks(value: float, device="cpu", group=None) -> float:
    """Timing rule of the bench: a multi-GPU number is the max over ranks."""
    import torch.distributed as dist
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    return float(t.item())


def rank_workload(wl, rank: int, world: int, kv_bytes_per_token: int = 1):
    """(task indices of this rank, full assignment) for a ``synth.Workload``."""
    costs = [task_cost(t, kv_bytes_per_token) for t in wl.tasks]
    assignment = assign_tasks(costs, world)
    return assignment[rank], assignment
