"""Multi-GPU sharding of the sampling-based planner ("running five independent controllers in parallel
and selecting the best control sequence at each step").

The controllers are independent until the final selection, so the path shards by CONTROLLERS: rank r runs its own
n_ctrl controllers over the global worlds [r * n_ctrl * worlds_per_ctrl, ...) (Philox is keyed by the global world index,
so the rollouts of a controller do not depend on which rank runs it).  The single exchange step of the whole path is
here: every rank contributes one row (score of its best controller, that controller's GLOBAL index, its plan:
2 + 4 H floats, 408 bytes at H = 25) to ONE all_gather -- NCCL on GPUs, gloo in the CPU test -- and every rank picks the
same winner (reading R31).

This module holds the collective and argument marshalling only: the row is packed by cf_mppi_pack_best and the winner
is picked by cf_mppi_select, both kernels of the library (cf.Sim.mppi_pack_best / mppi_select).
"""
from __future__ import annotations


def gather_rows(row, group=None):
    """All ranks' rows, stacked in rank order: [world][2 + 4 H] on the device of `row`.  The planner's one collective."""
    import torch
    import torch.distributed as dist
    if not dist.is_initialized():
        return row[None].contiguous()
    world = dist.get_world_size(group)      # (a group of one rank still goes through the collective)
    parts = [torch.empty_like(row) for _ in range(world)]
    dist.all_gather(parts, row.contiguous(), group=group)
    return torch.stack(parts)


def select_global_plan(sim, mp, out, rank: int, group=None):
    """out: the dict of cf.Sim.mppi_iterate on this rank.  Returns (plan [H][4], score, global controller index) as device
    tensors, identical on every rank.  No host synchronisation."""
    import torch
    row = sim.mppi_pack_best(mp, out["info"], out["plan"], rank * sim.params.n_ctrl)
    best = sim.mppi_select(gather_rows(row, group), mp.horizon)
    return best[2:].reshape(-1, 4), best[0], best[1].to(torch.int64)
