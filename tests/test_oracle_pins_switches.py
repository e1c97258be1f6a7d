"""Pins for the oracle parts VERDICT r1 found unpinned: the disturbance step (C8 step 4), the PARAM
slot map of both models (reading R17), the torque interface, the simplified abstracted model
 and the thrust-polynomial inverse of the mixer ("second-order polynomial").

None of them re-types an oracle formula: they are Newton's second law on a force-free body, statistics of the uniform
distribution, the (separately pinned, by r x f geometry) mixing matrix used as the inverse's check, and Eq. (8) at a
level attitude.  The Philox words, the uniform map and Box-Muller used to rebuild the expected draws are pinned on
their own in tests/test_oracle_pins.py (Random123 known answers, exact rationals, moments).
"""
import math

import numpy as np
import pytest
from scipy.spatial.transform import Rotation

M_, G_ = 0.027, 9.81
KF, KM = 3.16e-10, 7.94e-12
STREAM_PARAM, STREAM_DIST = 1, 2


def normals(cfo, seed, w, n, s, stream):
    x = cfo.philox(seed, (w, n, s, stream))
    z0, z1 = cfo.normal_pair(int(x[0]), int(x[1]))
    z2, z3 = cfo.normal_pair(int(x[2]), int(x[3]))
    return np.array([z0, z1, z2, z3])


# ---------------------------------------------------------------------------------- (a) disturbance step
def _dist_sim(cfo, integ, M, N, seed, sigma, offset=0, model=0):
    """A body no other force acts on: g = 0, rotors at rest with a zero command (FP) / zero thrust (AB), tilted, so that
    m dv/dt = f_dist exactly; the per-world mass is jittered over [0.8, 1.5] x nominal."""
    lo, hi = [1.0] * 12, [1.0] * 12
    lo[0], hi[0] = 0.8, 1.5
    ov = dict(integrator=integ, iface=cfo.IF_ROTOR if model == 0 else cfo.IF_ATTITUDE, g=0.0, dist_sigma=sigma,
              rnd_lo=lo, rnd_hi=hi, world_offset=offset)
    sim = cfo.OracleSim(M, N, model, ov)
    sim.reset(seed)
    q = Rotation.from_euler("xyz", [0.4, -0.3, 0.7])
    D = 17 if model == 0 else 13
    x = np.zeros((D, M * N))
    x[2] = 1.0
    if model == 0:
        x[3:7] = q.as_quat()[:, None]
    else:
        x[3:6] = np.array([0.4, -0.3, 0.7])[:, None]
    sim.set_full(state=x, step_counter=0)
    return sim


@pytest.mark.parametrize("model", [0, 1])
def test_disturbance_is_sigma_times_three_normals_of_the_dist_stream_in_the_world_frame(cfo, model):
    """C8 step (4): f_dist = sigma (z0, z1, z2) of Philox(seed; global world, drone, global step s, DIST), world frame,
    acting on the per-world mass: from rest with no other force one Euler step gives  v m_w / h = f_dist  exactly."""
    M, N, seed, sigma, off = 64, 3, 0xABCDEF0123, 0.005, 1000
    h = 1e-3 if model == 0 else 2e-3
    vi = 7 if model == 0 else 6
    sim = _dist_sim(cfo, 0, M, N, seed, sigma, off, model)
    m_w = np.repeat(sim.world_params()[0], N)
    assert m_w.std() > 0.1 * M_                                    # the masses really differ
    zero = np.zeros((3, M * N, 4), dtype=np.float32)
    rec = sim.step(zero, 3, cmd_hold=1, record_every=1)
    v_prev = np.zeros((3, M * N))
    for k in range(3):                                             # step k draws with index s = k
        want = np.array([sigma * normals(cfo, seed, w + off, n, k, STREAM_DIST)[:3] for w in range(M) for n in range(N)]).T
        got = (rec[k, vi:vi + 3] - v_prev) * m_w / h
        np.testing.assert_allclose(got, want, rtol=1e-9, atol=1e-15)
        v_prev = rec[k, vi:vi + 3]
    # a later global step: the index is the simulator's step counter, not the step within the call
    sim = _dist_sim(cfo, 0, M, N, seed, sigma, off, model)
    x0 = sim.get_state()
    sim.set_full(state=x0, step_counter=4242)
    sim.step(zero[:1], 1)
    want = np.array([sigma * normals(cfo, seed, w + off, n, 4242, STREAM_DIST)[:3] for w in range(M) for n in range(N)]).T
    np.testing.assert_allclose(sim.get_state()[vi:vi + 3] * m_w / h, want, rtol=1e-9, atol=1e-15)
    # neither the fourth normal nor the next step's draw is what is applied
    other = np.array([sigma * normals(cfo, seed, w + off, n, 4243, STREAM_DIST)[:3] for w in range(M) for n in range(N)]).T
    assert np.abs(sim.get_state()[vi:vi + 3] * m_w / h - other).max() > 1e-4


def test_disturbance_variance_and_hold_over_rk4_stages(cfo):
    """Sample variance of dv over many worlds = (sigma h / m)^2; the draw is held over the four RK4 stages: with a
    constant force RK4 and Euler give the same dv, and RK4 adds the exact h^2/2 a to the position."""
    M, seed, sigma, h = 4096, 11, 0.005, 1e-3
    lo = hi = [1.0] * 12
    ov = dict(iface=cfo.IF_ROTOR, g=0.0, dist_sigma=sigma, rnd_lo=lo, rnd_hi=hi)
    out = {}
    for integ in (0, 1):
        sim = cfo.OracleSim(M, 1, 0, dict(ov, integrator=integ))
        sim.reset(seed)
        x = np.zeros((17, M)); x[6] = 1.0
        sim.set_full(state=x, step_counter=0)
        sim.step(np.zeros((1, M, 4), dtype=np.float32), 1)
        out[integ] = sim.get_state()
    dv = out[0][7:10]
    n = dv.size
    var = (dv ** 2).mean() / (sigma * h / M_) ** 2                 # zero-mean: E z^2 = 1, Var z^2 = 2
    assert abs(var - 1) < 4 * math.sqrt(2 / n), var
    assert abs(dv.mean()) / (sigma * h / M_) < 4 / math.sqrt(n)
    assert abs(np.corrcoef(dv[0], dv[1])[0, 1]) < 4 / math.sqrt(M)  # three different normals, not one repeated
    np.testing.assert_allclose(out[1][7:10], dv, rtol=1e-12, atol=1e-18)
    np.testing.assert_allclose(out[1][0:3], 0.5 * h * dv, rtol=1e-12, atol=1e-18)
    assert np.all(out[0][0:3] == 0.0)                              # Euler: p+ = p + h v(old) = 0


# ---------------------------------------------------------------------------------- (b) PARAM slot map
FP_PLANES = {0: [0], 1: [1], 2: [2], 3: [3], 4: [4, 5, 6], 5: [7, 8, 9], 6: [10, 11, 12, 13], 7: [], 8: [], 9: [], 10: [], 11: []}
AB_PLANES = {0: [0], 1: [1], 2: [2], 3: [3], 4: [4], 5: [5], 6: [6], 7: [], 8: [7], 9: [8], 10: [9], 11: [10]}


@pytest.mark.parametrize("model", [0, 1])
def test_param_slots_one_at_a_time(cfo, model):
    """Reading R17 / cf.h: jitter on exactly one slot moves exactly the documented planes of world_params(), by the
    factor lo + (hi - lo) u with u the slot's word of Philox(seed; world, 0, block = slot // 4, PARAM)."""
    M, seed, lo_, hi_ = 3000, 77, 0.6, 1.9
    ov0 = dict(kf=[1e-3, 2e-7, KF], km=[1e-5, 3e-9, KM], cv_up=30.0, cv_dn=20.0, cd_up=1e-4, cd_dn=2e-4) if model == 0 else \
        dict(ab_a=[-130, -120, -110], ab_b=[-16, -15, -14], ab_c=[130, 120, 110], ab_ctau=33.0)
    base = cfo.OracleSim(M, 1, model, ov0)
    base.reset(seed)
    nominal = base.world_params()
    assert np.all(nominal == nominal[:, :1]) and np.all(nominal != 0)       # no jitter: every world at the nominal
    planes = FP_PLANES if model == 0 else AB_PLANES
    for slot in range(12):
        lo, hi = [1.0] * 12, [1.0] * 12
        lo[slot], hi[slot] = lo_, hi_
        sim = cfo.OracleSim(M, 1, model, dict(ov0, rnd_lo=lo, rnd_hi=hi))
        sim.reset(seed)
        wp = sim.world_params()
        moved = [j for j in range(wp.shape[0]) if not np.array_equal(wp[j], nominal[j])]
        assert moved == planes[slot], (model, slot, moved)
        if not moved:
            continue
        u = np.array([cfo.uniform(int(cfo.philox(seed, (w, 0, slot // 4, STREAM_PARAM))[slot % 4])) for w in range(M)])
        fac = lo_ + (hi_ - lo_) * u
        for j in moved:
            ratio = wp[j] / nominal[j]
            if model == 0 and slot == 6:        # the motor TIME constant is jittered: the rate coefficients divide
                ratio = 1.0 / ratio
            np.testing.assert_allclose(ratio, fac, rtol=1e-13)
        assert lo_ <= fac.min() and fac.max() <= hi_
        assert abs(fac.mean() - (lo_ + hi_) / 2) < 4 * (hi_ - lo_) / math.sqrt(12 * M)
        assert abs(fac.std() - (hi_ - lo_) / math.sqrt(12)) < 0.02


def test_ab_param_planes_are_the_coefficients_the_model_uses(cfo):
    """The planes the slot map names (a: 1-3, b: 4-6, c: 7-9, c_tau: 10) are the a, b, c, c_tau of Eqs. (9), (10): with
    only one family jittered, one Euler step from a state that excites only that term moves as the plane says."""
    M, seed, h = 50, 5, 2e-3
    for fam, slots, plane0 in (("a", (1, 2, 3), 1), ("b", (4, 5, 6), 4), ("c", (8, 9, 10), 7)):
        lo, hi = [1.0] * 12, [1.0] * 12
        for s_ in slots:
            lo[s_], hi[s_] = 0.5, 1.5
        sim = cfo.OracleSim(M, 1, 1, dict(rnd_lo=lo, rnd_hi=hi))
        sim.reset(seed)
        wp = sim.world_params()
        x = np.zeros((13, M)); x[2] = 1.0; x[12] = M_ * G_
        cmd = np.zeros((1, M, 4), dtype=np.float32); cmd[..., 3] = np.float32(M_ * G_)
        if fam == "a":
            x[3:6] = np.array([0.1, -0.2, 0.3])[:, None]; drive = x[3:6].copy()
        elif fam == "b":
            x[9:12] = np.array([1.0, -2.0, 3.0])[:, None]; drive = x[9:12].copy()
        else:
            cmd[..., 0:3] = np.array([0.25, -0.125, 0.5], dtype=np.float32); drive = cmd[0, :, 0:3].T.astype(np.float64)
        before = x[9:12].copy()
        sim.set_full(state=x, step_counter=0)
        sim.step(cmd, 1)
        ddpsi = (sim.get_state()[9:12] - before) / h          # Eq. (10) with one term alive
        np.testing.assert_allclose(ddpsi, wp[plane0:plane0 + 3] * drive, rtol=1e-9)
    lo, hi = [1.0] * 12, [1.0] * 12
    lo[11], hi[11] = 0.5, 1.5
    sim = cfo.OracleSim(M, 1, 1, dict(rnd_lo=lo, rnd_hi=hi))
    sim.reset(seed)
    x = np.zeros((13, M)); x[12] = 0.1
    sim.set_full(state=x, step_counter=0)
    cmd = np.zeros((1, M, 4), dtype=np.float32); cmd[..., 3] = np.float32(0.3)
    sim.step(cmd, 1)
    np.testing.assert_allclose((sim.get_state()[12] - 0.1) / h, sim.world_params()[10] * (float(np.float32(0.3)) - 0.1), rtol=1e-9)


# ---------------------------------------------------------------------------------- (c) torque interface
def test_torque_interface_commands_reach_the_body_as_commanded(cfo):
    """PAPER.md:L330 "collective thrust and body torque": the command (tau_x, tau_y, tau_z, F) goes through the motor
    mixer at the fetch; when nothing clips, the mixing matrix (pinned by geometry) applied to the held rotor commands
    returns exactly (F, tau)."""
    rng = np.random.default_rng(3)
    M = 40
    sim = cfo.OracleSim(M, 1, 0, dict(iface=cfo.IF_TORQUE))
    sim.reset(1)
    cmd = np.zeros((1, M, 4), dtype=np.float32)
    cmd[0, :, 0:2] = rng.uniform(-4e-4, 4e-4, (M, 2)); cmd[0, :, 2] = rng.uniform(-3e-5, 3e-5, M)
    cmd[0, :, 3] = rng.uniform(0.2, 0.35, M)
    sim.step(cmd, 1)
    rpm = sim.ctrl()[10:14]
    assert rpm.min() > 1.0 and rpm.max() < 21699.0
    for i in range(M):
        F, tau = cfo.mix(sim.params, rpm[:, i])
        c = cmd[0, i].astype(np.float64)
        assert abs(F - c[3]) < 1e-14
        np.testing.assert_allclose(tau, c[0:3], rtol=1e-9, atol=1e-18)
    assert sim.counters()[1] == 0                          # no attitude-controller tick on this interface
    # the body really feels it: with the rotors AT the commanded speeds, Eq. (4) from rest gives dw = tau / J
    x = sim.get_state()
    x[3:7] = np.array([0, 0, 0, 1.0])[:, None]; x[7:13] = 0; x[13:17] = rpm
    sim.set_full(state=x, step_counter=0)
    sim.step(cmd, 1)
    J = np.array([1.395e-5, 1.395e-5, 2.173e-5])
    np.testing.assert_allclose(sim.get_state()[10:13] / 1e-3, cmd[0, :, 0:3].T.astype(np.float64) / J[:, None], rtol=1e-8)
    # clipped case: a torque far beyond the rotors' authority saturates the commands at the limits
    big = np.zeros((1, M, 4), dtype=np.float32); big[..., 0] = 1.0; big[..., 3] = 0.3
    sim.step(big, 1)
    r = sim.ctrl()[10:14]
    assert np.all(r[0:2] == 0.0) and np.all(r[2:4] == 21700.0)


# ---------------------------------------------------------------------------------- (d) simplified abstracted model
@pytest.mark.parametrize("integ", [0, 1])
def test_simplified_abstracted_model_has_no_thrust_lag(cfo, integ):
    """without thrust dynamics the commanded thrust acts directly, f_Sigma == f_cmd: a level drone
    accelerates with f_cmd / m - g, NOT with the stored f_Sigma, and the state component equals the command afterwards.
    With the lag (Eq. (9)) the same step uses the stored value."""
    h, f_state = 2e-3, 0.1
    fc = float(np.float32(0.4))
    x0 = np.zeros((13, 1)); x0[2] = 1.0; x0[12] = f_state
    cmd = np.array([[[0, 0, 0, fc]]], dtype=np.float32)
    res = {}
    for dyn in (0, 1):
        sim = cfo.OracleSim(1, 1, 1, dict(integrator=integ, ab_thrust_dyn=dyn))
        sim.reset(0)
        sim.set_full(state=x0, step_counter=0)
        sim.step(cmd, 1)
        res[dyn] = sim.get_state()[:, 0]
    assert abs(res[0][8] - h * (fc / M_ - G_)) < 1e-14
    assert res[0][12] == fc
    if integ == 0:
        assert abs(res[1][8] - h * (f_state / M_ - G_)) < 1e-14
        assert abs(res[1][12] - (f_state + h * (fc - f_state) / 0.03)) < 1e-15
    else:   # exact solution of the lag: f(t) = fc + (f0 - fc) e^{-t/tau}, v = integral of f/m - g
        tau = 0.03
        vz = (fc * h + (f_state - fc) * tau * (1 - math.exp(-h / tau))) / M_ - G_ * h
        assert abs(res[1][8] - vz) < 1e-7 and abs(res[1][8] - res[0][8]) > 1e-3
    # many steps: the simplified model is a point mass under constant force, z = z0 + (fc/m - g) t^2/2 (RK4 exact)
    if integ == 1:
        sim = cfo.OracleSim(1, 1, 1, dict(integrator=1, ab_thrust_dyn=0))
        sim.reset(0)
        sim.set_full(state=x0, step_counter=0)
        sim.step(cmd, 100, cmd_hold=100)
        t = 100 * h
        assert abs(sim.get_state()[2, 0] - (1.0 + 0.5 * (fc / M_ - G_) * t * t)) < 1e-12


# ---------------------------------------------------------------------------------- (e) thrust-polynomial inverse
def test_mixer_inverts_the_thrust_polynomial_with_its_positive_root(cfo):
    """rotor thrust is a SECOND-ORDER POLYNOMIAL of the rotor speed; the mixer must return the speed at
    which that polynomial gives the wanted thrust.  Checked through the mixing matrix (pinned by geometry): thrust sum
    and roll / pitch torque of the held rotor commands equal the command, every speed is the positive root."""
    kf = [2.0e-3, 1.5e-6, 2.4e-10]
    rng = np.random.default_rng(5)
    M = 60
    sim = cfo.OracleSim(M, 1, 0, dict(iface=cfo.IF_TORQUE, kf=kf))
    sim.reset(2)
    cmd = np.zeros((1, M, 4), dtype=np.float32)
    cmd[0, :, 0:2] = rng.uniform(-4e-4, 4e-4, (M, 2)); cmd[0, :, 3] = rng.uniform(0.2, 0.35, M)
    sim.step(cmd, 1)
    rpm = sim.ctrl()[10:14]
    assert rpm.min() > 1000.0 and rpm.max() < 21699.0
    lever = 0.046 / math.sqrt(2)
    for i in range(M):
        F, tau = cfo.mix(sim.params, rpm[:, i])
        c = cmd[0, i].astype(np.float64)
        assert abs(F - c[3]) < 1e-12
        np.testing.assert_allclose(tau[0:2], c[0:2], rtol=1e-9, atol=1e-16)
        f = kf[0] + kf[1] * rpm[:, i] + kf[2] * rpm[:, i] ** 2
        np.testing.assert_allclose(f.sum(), c[3], rtol=1e-12)
        # per rotor: thrust = F/4 -+ tau_x/(4 l) -+ tau_y/(4 l) on the X layout (rotor 1 at (+,-): both signs negative)
        assert abs(f[0] - (c[3] / 4 - c[0] / (4 * lever) - c[1] / (4 * lever))) < 1e-12
    # hover speed after a reset is the positive root as well: 4 f(W_hover) = m g
    wh = cfo.OracleSim(1, 1, 0, dict(kf=kf))
    wh.reset(0)
    W = wh.get_state()[13:, 0]
    assert np.all(W > 0) and abs(4 * (kf[0] + kf[1] * W[0] + kf[2] * W[0] ** 2) - M_ * G_) < 1e-14
