"""Multi-GPU sharding of the sampling-based planner ("running five independent controllers in parallel
and selecting the best control sequence at each step").

The controllers are independent until the final selection, so the path shards by CONTROLLERS: rank r runs its own
n_ctrl controllers over the global worlds [r * n_ctrl * worlds_per_ctrl, ...) (Philox is keyed by the global world index,
so the rollouts of a controller do not depend on which rank runs it) and the single exchange step of the whole path is
here: every rank contributes (score of its best controller, that controller's plan), H * 16 + 8 bytes, and all ranks
pick the same winner -- lowest score, ties to the lowest global controller index (reading R31).  One all_gather of a
[2 + 4 H] float32 row per planning iteration; NCCL on GPUs, gloo in the CPU test (tests/test_planner_gloo.py).

Argument marshalling and the collective only: the per-rank compute is cf_mppi_iterate (the CUDA path).
"""
from __future__ import annotations


def pack_local_best(info, plan, n_ctrl: int, rank: int):
    """info: float32 [4 n_ctrl + 4] of cf_mppi_update (device or CPU tensor), plan: [H][4] -> one row
    [score, global controller index, plan...] on the same device.  No host synchronisation."""
    import torch
    best = info[4 * n_ctrl:4 * n_ctrl + 1].view(torch.int32).to(torch.int64)            # local best controller
    score = info[0:4 * n_ctrl:4].gather(0, best)
    gidx = (best + rank * n_ctrl).to(torch.float32)                                      # exact: small integers
    return torch.cat([score, gidx, plan.reshape(-1)])


def select_global_plan(row, group=None):
    """row: this rank's pack_local_best(...).  Returns (plan [H][4], score, global controller index) -- identical on
    every rank.  The one collective of the planner path."""
    import torch
    import torch.distributed as dist
    world = dist.get_world_size(group) if dist.is_initialized() else 1
    if world == 1:
        rows = row[None]
    else:
        parts = [torch.empty_like(row) for _ in range(world)]
        dist.all_gather(parts, row.contiguous(), group=group)
        rows = torch.stack(parts)
    # lowest score wins; ties -> lowest global controller index (rows are in rank order = controller order)
    score = rows[:, 0]
    win = torch.argmin(torch.where(torch.isnan(score), torch.full_like(score, float("inf")), score))
    best = rows[win]
    return best[2:].reshape(-1, 4), best[0], best[1].to(torch.int64)
