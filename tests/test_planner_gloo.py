"""N > 1 path of the planner on CPU: two gloo ranks each run their own controllers (sharding
by controllers, global world indices via world_offset) and exchange one [2 + 4 H] row per iteration
(paper_2606_01478_b200/planner.py); every rank must end up with the plan a single process running all controllers selects.
The per-rank compute here is the oracle (no GPU in this container); on GPUs it is cf_mppi_iterate."""
import os
import socket
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
N_LOCAL, KC, H, HOLD, N_ELITE, LAM = 2, 48, 5, 4, 6, 0.3


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _local_update(rank, n_ctrl, seed=5):
    """oracle rollout + update of controllers [rank * n_ctrl, (rank + 1) * n_ctrl) -> (info like cf_mppi_update, plan)"""
    from oracle import cfo, mppi as omppi
    from paper_2606_01478_b200 import workloads as W
    wl = W.mppi(seed=seed, n_ctrl=n_ctrl, worlds_per_ctrl=KC, horizon=H, cmd_hold=HOLD, n_elite=N_ELITE)
    off = rank * n_ctrl * KC
    p = dict(wl.params, world_offset=off)
    nominal = wl.cmds.copy()
    nominal[..., 0] = 0.05 * (rank * n_ctrl + np.arange(n_ctrl))[:, None]      # a different nominal per GLOBAL controller
    sim = cfo.OracleSim(wl.M, 1, wl.model, p)
    sim.reset(wl.seed)
    sim.set_state(wl.broadcast_state, broadcast=True)
    sim.step(nominal, wl.n_steps, cmd_hold=HOLD)
    out = omppi.update(sim.cost().astype(np.float32), nominal, seed=wl.seed, world_offset=off,
                       worlds_per_ctrl=KC, s_start=0, cmd_hold=HOLD, sigma=p["noise_sigma"], beta=p["noise_beta"],
                       lo=p["cmd_lo"], hi=p["cmd_hi"], n_elite=N_ELITE, lam=LAM, shift=1)
    info = np.zeros(4 * n_ctrl + 4, dtype=np.float32)
    info[0:4 * n_ctrl:4] = out["score"]
    info[4 * n_ctrl:4 * n_ctrl + 1] = np.array([out["best"]], dtype=np.int32).view(np.float32)
    return info, out["plan"].astype(np.float32), out


def _pack(info, plan, n_ctrl, rank):
    """the row cf_mppi_pack_best writes, restated for the CPU run: [score of the local best, GLOBAL controller index, plan]"""
    best = int(info[4 * n_ctrl:4 * n_ctrl + 1].view(np.int32)[0])
    return np.concatenate([[info[4 * best], np.float32(best + rank * n_ctrl)], plan.reshape(-1)]).astype(np.float32)


def _worker(rank, world, port, out_path):
    sys.path.insert(0, ROOT)
    import torch
    import torch.distributed as dist
    from oracle import cfo, mppi as omppi
    from paper_2606_01478_b200 import planner
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    cfo.set_num_threads(1)
    info, plan, _ = _local_update(rank, N_LOCAL)
    rows = planner.gather_rows(torch.from_numpy(_pack(info, plan, N_LOCAL, rank))).numpy()    # the product's collective
    assert rows.shape == (world, 2 + 4 * H) and rows[rank, 1] >= rank * N_LOCAL               # rank order
    best = rows[omppi.select_rows(rows)]                                                       # R31 by the oracle
    gplan = torch.from_numpy(best[2:].reshape(-1, 4).copy())
    gathered = [torch.empty_like(gplan) for _ in range(world)]
    dist.all_gather(gathered, gplan)
    assert all(torch.equal(g, gplan) for g in gathered)            # every rank holds the same plan
    if rank == 0:
        np.savez(out_path, plan=gplan.numpy(), score=float(best[0]), gidx=int(best[1]))
    dist.destroy_process_group()


def test_two_ranks_select_the_plan_of_the_single_process_run(tmp_path):
    import torch.multiprocessing as mp
    sys.path.insert(0, ROOT)
    out = str(tmp_path / "plan.npz")
    mp.start_processes(_worker, args=(2, _free_port(), out), nprocs=2, join=True, start_method="spawn")
    got = np.load(out)
    # single process: all four controllers at once
    _, _, ref = _local_update(0, 2 * N_LOCAL)
    assert int(got["gidx"]) == ref["best"]
    assert np.array_equal(got["plan"], ref["plan"].astype(np.float32))
    assert got["score"] == np.float32(ref["score"][ref["best"]])


def test_row_selection_rule_ties_and_nan():
    """R31 across shards (oracle side; the library's cf_mppi_select is held to it in tests/test_gpu_mppi.py): lowest score,
    ties -> lowest global controller index whatever the row order, NaN never wins, -0.0 < +0.0 in the total order."""
    sys.path.insert(0, ROOT)
    from oracle import mppi as omppi
    H_ = 2
    def row(score, idx):
        return np.concatenate([[score, idx], np.full(4 * H_, idx)]).astype(np.float32)
    assert omppi.select_rows([row(3.0, 6), row(3.0, 2), row(5.0, 0)]) == 1
    assert omppi.select_rows([row(np.nan, 0), row(7.0, 3)]) == 1
    assert omppi.select_rows([row(0.0, 0), row(-0.0, 1)]) == 1
    assert omppi.select_rows([row(np.nan, 4), row(np.nan, 1)]) == 1
    assert omppi.select_rows([row(-1.0, 9)]) == 0
    info = np.zeros(12, dtype=np.float32)
    info[0:8:4] = [4.0, 3.0]
    info[8:9] = np.array([1], dtype=np.int32).view(np.float32)
    r = _pack(info, np.arange(8, dtype=np.float32).reshape(2, 4), 2, rank=3)
    assert r[0] == 3.0 and r[1] == 7.0 and np.array_equal(r[2:], np.arange(8))
