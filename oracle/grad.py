"""float64 ORACLE for the gradient workload of PAPER.md:L63/L69 (Fig. 3D): "differentiating a goal distance with respect
to the control inputs" through n consecutive simulation steps (dynamics AND onboard controller stack).

TEST INFRASTRUCTURE ONLY (see oracle/cfo.h).  Shares nothing with paper_2606_01478_b200/.

The quantity has a plain definition, so the oracle is that definition written out: with the simulator state x_0 fixed,

    L(u) = || p_n(u) - goal ||,      p_n = position after n steps of the float64 oracle step (oracle/cfo.c) driven by the
                                     command sequence u[k], k = 0..K-1, each held cmd_hold steps,
    g[k][j] = dL / du[k][j]          taken as a central finite difference of the oracle's forward map, Richardson-
                                     extrapolated:  D(h) = (L(u + h e) - L(u - h e)) / 2h,  g = (4 D(h/2) - D(h)) / 3,

which is the derivative of the map wherever it is differentiable (error O(h^4) + rounding ~1e-10 relative at h = 1e-4 of
the command scale).  At the kinks of the method (actuator / integral clipping, C5-C7) the derivative does not exist and
the comparison is made away from them (R33); hard saturation, where the map is locally constant, is compared
too.  Worlds are independent, so one perturbed run differentiates the same input of every world at once: 4 runs per
(k, j).  The commands are float32 inputs of the step (both sides see the same bits), so the perturbation is applied to a
float64 copy through cfo_step_f64cmd -- see `forward`.

Pins: tests/test_oracle_grad.py (closed forms of linear channels via matrix powers, a hand-derived three-step chain
through mixer, motor lag and thrust curve, symmetry / zero-gradient cases).
"""
from __future__ import annotations

import numpy as np

from . import cfo

# perturbation per command component (roll, pitch, yaw [rad], thrust [N]; rotor interface: rpm)
STEP_ATT = np.array([1e-3, 1e-3, 1e-3, 1e-3])
STEP_RPM = np.array([20.0, 20.0, 20.0, 20.0])


class Snapshot:
    """Everything a step depends on, so that every forward run starts from the same simulator state."""

    def __init__(self, sim: cfo.OracleSim):
        self.state, self.ctrl = sim.get_state(), sim.ctrl()
        self.wparam, self.mind2 = sim.world_params(), sim.min_d2()
        self.s = int(sim.counters()[0])

    def restore(self, sim: cfo.OracleSim):
        sim.set_full(state=self.state, ctrl=self.ctrl, wparam=self.wparam, mind2=self.mind2, step_counter=self.s)


def forward(sim: cfo.OracleSim, snap: Snapshot, cmds64: np.ndarray, n_steps: int, cmd_hold: int, goal) -> np.ndarray:
    """L(u) for every drone: [MN].  cmds64: float64 [K][MN][4] (exact, not rounded to float32)."""
    snap.restore(sim)
    sim.step_f64(cmds64, n_steps, cmd_hold=cmd_hold)
    p = sim.get_state()[:3]
    return np.sqrt(((p - np.asarray(goal, dtype=np.float64).reshape(3, 1)) ** 2).sum(0))


def value_and_grad(sim: cfo.OracleSim, cmds, n_steps: int, cmd_hold: int, goal, steps=None):
    """Returns (L [MN], g [K][MN][4]) at the simulator's current state, which is left unchanged."""
    cm = np.ascontiguousarray(cmds, dtype=np.float32).astype(np.float64).reshape(-1, sim.MN, 4)
    K = cm.shape[0]
    if steps is None:
        steps = STEP_RPM if sim.params.iface == cfo.IF_ROTOR else STEP_ATT
    snap = Snapshot(sim)
    L0 = forward(sim, snap, cm, n_steps, cmd_hold, goal)
    g = np.zeros((K, sim.MN, 4))
    for k in range(K):
        if k * cmd_hold >= n_steps:
            continue                                  # command never used
        for j in range(4):
            D = []
            for h in (steps[j], 0.5 * steps[j]):
                up, dn = cm.copy(), cm.copy()
                up[k, :, j] += h
                dn[k, :, j] -= h
                D.append((forward(sim, snap, up, n_steps, cmd_hold, goal)
                          - forward(sim, snap, dn, n_steps, cmd_hold, goal)) / (2 * h))
            g[k, :, j] = (4 * D[1] - D[0]) / 3
    snap.restore(sim)
    return L0, g
