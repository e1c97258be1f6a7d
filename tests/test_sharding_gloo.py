"""N > 1 path on CPU: two gloo ranks each simulate their contiguous shard of worlds (world_offset), with no data-path
collective; gathering the shards reproduces the single-process run bit-exactly.  The per-rank
simulator here is the oracle (there is no GPU in this container); the GPU equivalent is
tests/test_gpu_parity.py::test_world_offset_shards_reproduce_the_full_run."""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, name, kw, out_path):
    sys.path.insert(0, ROOT)
    import torch
    import torch.distributed as dist
    from oracle import cfo
    from paper_2606_01478_b200 import workloads as W
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    cfo.set_num_threads(1)
    wl = W.make(name, **kw)
    lo, m = W.shard_worlds(wl.M, world, rank)
    sim = cfo.OracleSim(m, wl.N, wl.model, dict(wl.params, world_offset=lo))
    sim.reset(wl.seed)
    if wl.broadcast_state is not None:
        sim.set_state(wl.broadcast_state, broadcast=True)
    cm = wl.cmds if wl.cmds.ndim == 2 else wl.cmds[:, lo * wl.N:(lo + m) * wl.N]
    dist.barrier()
    sim.step(cm, wl.n_steps, cmd_hold=wl.cmd_hold)
    dist.barrier()
    # timing reduction used by bench.py: max over ranks
    t = torch.tensor([float(rank + 1)], dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    assert t.item() == world
    x = torch.from_numpy(sim.get_state())                      # [D][m*N]
    sizes = [W.shard_worlds(wl.M, world, r)[1] * wl.N for r in range(world)]
    parts = [torch.empty((wl.D, n), dtype=torch.float64) for n in sizes]
    if len(set(sizes)) == 1:
        dist.all_gather(parts, x)
    else:                                                      # ragged shards: gather by broadcast
        for r in range(world):
            if r == rank:
                parts[r].copy_(x)
            dist.broadcast(parts[r], src=r)
    if rank == 0:
        np.save(out_path, torch.cat(parts, dim=1).numpy())
    dist.destroy_process_group()


@pytest.mark.parametrize("name,kw", [("cfg5", dict(M=37, n_steps=25, seed=3)), ("cfg3", dict(M=64, n_steps=20, seed=3)),
                                     ("cfg4", dict(M=4, N=9, n_steps=30, seed=3))])
def test_two_gloo_ranks_reproduce_single_run(tmp_path, cfo, name, kw):
    import torch.multiprocessing as mp
    from paper_2606_01478_b200 import workloads as W
    out = str(tmp_path / "gathered.npy")
    mp.spawn(_worker, args=(2, _free_port(), name, kw, out), nprocs=2, join=True)
    wl = W.make(name, **kw)
    sim = cfo.OracleSim(wl.M, wl.N, wl.model, wl.params)
    sim.reset(wl.seed)
    if wl.broadcast_state is not None:
        sim.set_state(wl.broadcast_state, broadcast=True)
    sim.step(wl.cmds, wl.n_steps, cmd_hold=wl.cmd_hold)
    assert np.array_equal(np.load(out), sim.get_state())


def test_shard_worlds_partition():
    from paper_2606_01478_b200 import workloads as W
    for M in (1, 7, 64, 1000, 1 << 20):
        for ws in (1, 2, 3, 8):
            parts = [W.shard_worlds(M, ws, r) for r in range(ws)]
            assert parts[0][0] == 0 and sum(m for _, m in parts) == M
            for (lo, m), (lo2, _) in zip(parts, parts[1:]):
                assert lo + m == lo2
            assert max(m for _, m in parts) - min(m for _, m in parts) <= 1
