"""Helpers shared by the CPU (oracle) and GPU (parity) tests.  No method arithmetic here."""
import numpy as np


def split_calls(wl, chunks):
    """Cut wl's run into successive step() calls: yields (cmds, n_steps, cmd_hold).  Every call stays inside one
    command segment (or, for cmd_hold == 1, takes its own slice), so the held command is the same as in the
    fused run: the command index of a step is (s - s0) // cmd_hold relative to the call."""
    t, ci = 0, 0
    while t < wl.n_steps:
        n = min(chunks[ci % len(chunks)], wl.n_steps - t)
        if wl.cmd_hold == 1:
            yield wl.cmds[t:t + n], n, 1
        else:
            k0 = t // wl.cmd_hold
            n = min(n, wl.cmd_hold - t % wl.cmd_hold)
            yield wl.cmds[k0:k0 + 1], n, n
        t += n
        ci += 1


def fresh_oracle(cfo, wl, **extra):
    sim = cfo.OracleSim(wl.M, wl.N, wl.model, dict(wl.params, **extra))
    sim.reset(wl.seed)
    if wl.broadcast_state is not None:
        sim.set_state(wl.broadcast_state, broadcast=True)
    return sim
