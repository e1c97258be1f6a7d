"""Pins of the gradient oracle (oracle/grad.py; Fig. 3D: goal distance differentiated w.r.t. the control
inputs through n steps).  The oracle is a finite difference of the float64 step; these checks fix it from outside:
closed forms of the linear vertical channel (matrix powers / the RK4 amplification polynomial, built here in numpy),
a hand-derived three-step chain through mixer, motor lag and thrust curve, symmetry zeros, hard saturation, and
convergence of the difference quotient on a generic closed-loop case.
"""
import math

import numpy as np
import pytest

M_, G_ = 0.027, 9.81
KF = 3.16e-10
W_HOVER = math.sqrt(M_ * G_ / (4 * KF))
HOVER = float(np.float32(M_ * G_))


@pytest.fixture(scope="module")
def og():
    from oracle import grad
    return grad


def ab_sim(cfo, integrator, f_phys=500.0):
    sim = cfo.OracleSim(1, 1, cfo.MODEL_AB, dict(integrator=integrator, iface=cfo.IF_ATTITUDE, f_phys=f_phys,
                                                 f_att=f_phys, init_mode=0))
    sim.reset(1)
    return sim


def vertical_channel(h, integrator, ctau=1 / 0.03):
    """x = (z, vz, f);  dx/dt = Ac x + Bc u + const.  One step: x+ = Phi x + Gam u + const."""
    Ac = np.array([[0, 1, 0], [0, 0, 1 / M_], [0, 0, -ctau]])
    Bc = np.array([0, 0, ctau])
    if integrator == 0:
        return np.eye(3) + h * Ac, h * Bc
    hA = h * Ac
    Phi = np.eye(3) + hA + hA @ hA / 2 + hA @ hA @ hA / 6 + hA @ hA @ hA @ hA / 24
    Gam = h * (np.eye(3) + hA / 2 + hA @ hA / 6 + hA @ hA @ hA / 24) @ Bc
    return Phi, Gam


@pytest.mark.parametrize("integrator", [0, 1])
@pytest.mark.parametrize("hold", [1, 3])
def test_linear_vertical_channel_matches_matrix_power_closed_form(cfo, og, integrator, hold):
    n, h = 12, 1 / 500.0
    K = n // hold
    sim = ab_sim(cfo, integrator)
    x0 = np.zeros(13); x0[2] = 1.0; x0[8] = 0.3; x0[12] = 0.9 * HOVER
    sim.set_state(x0, broadcast=True)
    rng = np.random.default_rng(0)
    cmds = np.zeros((K, 1, 4), dtype=np.float32)
    cmds[:, 0, 3] = HOVER + rng.uniform(-0.05, 0.05, K)
    goal = np.array([0.4, -0.3, 1.5])                  # e_x, e_y stay (-0.4, 0.3): level flight never moves sideways
    L, g = og.value_and_grad(sim, cmds, n, hold, goal)
    Phi, Gam = vertical_channel(h, integrator)
    # z_n sensitivity to the command of step s: [Phi^(n-1-s) Gam]_z ; a held command sums its steps
    dz = np.array([sum(np.linalg.matrix_power(Phi, n - 1 - s) @ Gam for s in range(k * hold, (k + 1) * hold))[0]
                   for k in range(K)])
    z_n = sim_final_z(cfo, sim, cmds, n, hold)
    e = np.array([0.0 - goal[0], 0.0 - goal[1], z_n - goal[2]])
    assert L[0] == pytest.approx(np.linalg.norm(e), rel=1e-12)
    np.testing.assert_allclose(g[:, 0, 3], e[2] / np.linalg.norm(e) * dz, rtol=2e-7, atol=2e-12)
    assert np.abs(g[:, 0, 2]).max() < 1e-9             # yaw command: no effect on the position of a level drone
    assert np.abs(g[:, 0, :2]).max() < 1e-6 * np.abs(g[:, 0, 3]).max() + 1e-3   # roll / pitch: first order only in x, y
    # the state was left untouched
    assert np.array_equal(sim.get_state()[:, 0], x0)


def sim_final_z(cfo, sim, cmds, n, hold):
    from oracle import grad
    snap = grad.Snapshot(sim)
    sim.step(cmds, n, cmd_hold=hold)
    z = sim.get_state()[2, 0]
    snap.restore(sim)
    return z


def test_roll_command_moves_the_drone_sideways_with_the_sign_of_reading_r13(cfo, og):
    """R = Rz Ry Rx: positive roll tilts thrust towards -y, positive pitch towards +x (z_B of C3)."""
    sim = ab_sim(cfo, 0)
    n = 20
    cmds = np.zeros((n, 1, 4), dtype=np.float32); cmds[..., 3] = HOVER
    goal_y = np.array([0.0, -5.0, 1.0])                # far away on -y: L = distance, dL/dy = +1 ... moving to -y lowers L
    _, g = og.value_and_grad(sim, cmds, n, 1, goal_y)
    assert (g[:-3, 0, 0] < 0).all()                    # more roll -> closer to the goal on -y
    goal_x = np.array([5.0, 0.0, 1.0])
    _, g = og.value_and_grad(sim, cmds, n, 1, goal_x)
    assert (g[:-3, 0, 1] < 0).all()                    # more pitch -> closer to the goal on +x
    assert np.abs(g[-1]).max() == 0.0                  # the last command cannot reach the position in one Euler step


def test_hand_derived_three_step_chain_through_mixer_lag_and_thrust_curve(cfo, og):
    h, tau = 1e-3, 0.03
    sim = cfo.OracleSim(1, 1, cfo.MODEL_FP, dict(integrator=cfo.EULER, iface=cfo.IF_ATTITUDE, f_phys=1000.0,
                                                 f_att=500.0, init_mode=0))
    sim.reset(1)                                       # level hover at (0,0,1), rotors at hover speed
    F = np.float32(0.30)
    cmds = np.zeros((1, 1, 4), dtype=np.float32); cmds[0, 0, 3] = F
    goal = np.array([0.0, 0.0, 3.0])                   # straight above: L = 3 - z_3
    L, g = og.value_and_grad(sim, cmds, 3, 3, goal)
    # s=0: tick -> W_cmd = sqrt(F / 4 kf); W1 = W0 + (h/tau)(W_cmd - W0).  s=1 (no tick, att_div = 2): v2 = v1 + h (4 kf W1^2/m - g).
    # s=2: p3 = p2 + h v2.  z3 depends on F only through v2 <- W1 <- W_cmd:
    w_cmd = math.sqrt(float(F) / (4 * KF))
    w1 = W_HOVER + (h / tau) * (w_cmd - W_HOVER)
    dz3_dF = h * h * (8 * KF * w1 / M_) * (h / tau) * (1.0 / (8 * KF * w_cmd))
    assert g[0, 0, 3] == pytest.approx(-dz3_dF, rel=1e-6)
    assert np.abs(g[0, 0, :3]).max() < 1e-12           # level, goal on the axis: attitude commands act at second order
    z3 = 1.0 + h * (h * (4 * KF * W_HOVER ** 2 / M_ - G_)) + h * (h * (4 * KF * W_HOVER ** 2 / M_ - G_) + h * (4 * KF * w1 ** 2 / M_ - G_))
    assert L[0] == pytest.approx(3.0 - z3, rel=1e-12)


def test_hard_saturation_has_zero_gradient_and_rotor_interface_is_differentiated_in_rpm(cfo, og):
    sim = cfo.OracleSim(2, 1, cfo.MODEL_FP, dict(integrator=cfo.RK4, iface=cfo.IF_ATTITUDE, f_phys=1000.0, f_att=500.0,
                                                 init_mode=0))
    sim.reset(1)
    cmds = np.zeros((2, 2, 4), dtype=np.float32)
    cmds[:, 0, 3] = 2.0                                # world 0: far beyond 4 x 0.1488 N: every rotor clipped
    cmds[:, 1, 3] = 0.3
    _, g = og.value_and_grad(sim, cmds, 8, 4, [0.0, 0.0, 3.0])
    assert np.abs(g[:, 0, :]).max() == 0.0
    assert (g[0, 1, 3] < 0) and g[1, 1, 3] < 0
    rot = cfo.OracleSim(1, 1, cfo.MODEL_FP, dict(integrator=cfo.EULER, iface=cfo.IF_ROTOR, f_phys=1000.0, init_mode=0))
    rot.reset(1)
    rc = np.full((1, 1, 4), W_HOVER + 500.0, dtype=np.float32)
    _, g = og.value_and_grad(rot, rc, 3, 3, [0.0, 0.0, 3.0])
    w1 = W_HOVER + (1e-3 / 0.03) * (float(rc[0, 0, 0]) - W_HOVER)
    per_rotor = 1e-3 * 1e-3 * (2 * KF * w1 / M_) * (1e-3 / 0.03)      # same chain, one rotor, no mixer
    np.testing.assert_allclose(g[0, 0], -per_rotor, rtol=1e-6)


def test_difference_quotient_has_converged_on_a_generic_closed_loop_case(cfo, og):
    """FP, RK4, attitude controller active, tilted start, 10 steps (the Fig. 3D shape): the extrapolated quotient does
    not depend on the step size, and it predicts a finite displacement of the commands to second order."""
    sim = cfo.OracleSim(6, 1, cfo.MODEL_FP, dict(integrator=cfo.RK4, iface=cfo.IF_ATTITUDE, f_phys=1000.0, f_att=500.0,
                                                 init_mode=1, p0_lo=[-1, -1, 0], p0_hi=[1, 1, 2], tilt0_max=0.4))
    sim.reset(5)
    rng = np.random.default_rng(2)
    cmds = np.zeros((10, 6, 4), dtype=np.float32)
    cmds[..., :2] = rng.uniform(-0.2, 0.2, (10, 6, 2)); cmds[..., 3] = rng.uniform(0.2, 0.35, (10, 6))
    goal = [0.5, -0.2, 1.2]
    L, g = og.value_and_grad(sim, cmds, 10, 1, goal)
    _, g2 = og.value_and_grad(sim, cmds, 10, 1, goal, steps=0.3 * og.STEP_ATT)
    np.testing.assert_allclose(g, g2, rtol=1e-5, atol=1e-11)      # rounding floor of the quotient: eps L / h
    d = rng.standard_normal(cmds.shape) * np.array([1e-3, 1e-3, 1e-3, 1e-4])
    snap = og.Snapshot(sim)
    Lp = og.forward(sim, snap, cmds.astype(np.float64) + d, 10, 1, goal)
    Lm = og.forward(sim, snap, cmds.astype(np.float64) - d, 10, 1, goal)
    np.testing.assert_allclose((Lp - Lm) / 2, (g * d).sum(axis=(0, 2)), rtol=1e-4)
    assert np.abs(g[0:8:2, :, 3]).min() > 0            # every early thrust command a controller tick sees matters ...
    assert np.abs(g[1::2]).max() == 0.0                # ... and the ones fetched between two 500 Hz ticks never act (C8)
