"""Round-3 pins of the float64 oracle for the three parts VERDICT r2 found unpinned: the thrust scaling coefficient c_f
of Eq. (8), the attitude-integral limit of the controller tick (C5, the "Mellinger control type" of
PAPER.md:L330; reading R7) and the component order of the Box-Muller pair (C9).  Same rules as test_oracle_pins.py:
closed forms, scipy rotations, hand-worked values -- a single-token mutation of oracle/cfo.c in any of the three places
(c_f dropped, c_f applied to Eq. (9) instead of Eq. (8), clip removed or one-sided, cos / sin swapped) fails one of them.
"""
import math

import numpy as np
import pytest
from scipy.spatial.transform import Rotation

from test_oracle_pins import G_, J_, M_, ab_state, cmd1, fp_state, rotor_sim

CF = 0.8


# ---------------------------------------------------------------------------------- Eq. (8): c_f scales the thrust force
def test_eq8_cf_level_stationary_thrust_is_mg_over_cf(cfo):
    """Level drone: m dv = c_f f_Sigma - m g = 0  <=>  f_Sigma = m g / c_f.  With f_Sigma = m g (stationary for c_f = 1)
    the drone falls with (c_f - 1) g."""
    f_eq = float(np.float32(M_ * G_ / CF))                       # float32-exact command = held thrust state: Eq. (9) is at rest
    sim = rotor_sim(cfo, 1, dict(ab_cf=CF), model=1)
    sim.set_full(state=ab_state(f=f_eq), step_counter=0)
    sim.step(cmd1([0, 0, 0, f_eq]), 250, cmd_hold=250)
    x = sim.get_state()[:, 0]
    t = 250 * 0.002
    az = CF * f_eq / M_ - G_                                      # float32 rounding of the command: ~1e-8 m/s^2, carried exactly
    assert abs(az) < 1e-6
    np.testing.assert_allclose(x[8], az * t, rtol=0, atol=1e-13)
    np.testing.assert_allclose(x[2], 1 + 0.5 * az * t * t, rtol=0, atol=1e-13)   # RK4: exact on a parabola
    assert x[12] == f_eq and np.all(x[[0, 1, 3, 4, 5, 6, 7]] == 0)
    mg = float(np.float32(M_ * G_))
    sim.set_full(state=ab_state(f=mg), step_counter=0)
    sim.step(cmd1([0, 0, 0, mg]), 100, cmd_hold=100)
    assert abs(sim.get_state()[8, 0] - (CF * mg / M_ - G_) * 0.2) < 1e-13
    assert abs((CF * mg / M_ - G_) - (CF - 1) * G_) < 1e-6


def test_eq8_cf_tilted_one_euler_step_against_scipy_and_eq9_untouched(cfo):
    """One Euler step from rest at attitude Psi: dv = h (R e_z c_f f_Sigma / m - g e_z), R = scipy 'xyz'; the thrust state
    follows Eq. (9) -- f + h c_tau (f_c - f) -- with NO c_f in it."""
    h = 1e-4
    sim = rotor_sim(cfo, 0, dict(f_phys=1e4, f_att=1e4, f_pos=1e4, ab_cf=CF), model=1)
    psi, f, fc = (0.3, -0.4, 0.9), 0.31, float(np.float32(0.25))
    sim.set_full(state=ab_state(psi=psi, f=f), step_counter=0)
    sim.step(cmd1([0, 0, 0, fc]), 1)
    x = sim.get_state()[:, 0]
    want = Rotation.from_euler("xyz", psi).apply([0, 0, CF * f / M_]) - [0, 0, G_]
    np.testing.assert_allclose(x[6:9] / h, want, rtol=1e-10, atol=1e-9)
    assert abs(x[12] - (f + h * (fc - f) / 0.03)) < 1e-15        # Eq. (9): c_tau = 1 / 0.03 s (defaults), independent of c_f
    # and over many steps the thrust lag is the closed form of P11 whatever c_f is
    sim2 = rotor_sim(cfo, 0, dict(ab_cf=CF), model=1)
    sim2.set_full(state=ab_state(f=0.1), step_counter=0)
    k, z = 80, 0.002 / 0.03
    fc2 = float(np.float32(0.3))
    sim2.step(cmd1([0, 0, 0, fc2]), k, cmd_hold=k)
    assert abs(sim2.get_state()[12, 0] - (fc2 + (0.1 - fc2) * (1 - z) ** k)) < 1e-15


def test_eq8_cf_simplified_model_scales_the_command(cfo):
    """PAPER.md:L354 simplified variant (no thrust state): the force is c_f f_cmd."""
    sim = rotor_sim(cfo, 0, dict(f_phys=1e4, f_att=1e4, f_pos=1e4, ab_cf=CF, ab_thrust_dyn=0), model=1)
    fc = float(np.float32(0.29))
    sim.set_full(state=ab_state(psi=(0.2, 0.1, -0.3), f=0.0), step_counter=0)
    sim.step(cmd1([0, 0, 0, fc]), 1)
    want = Rotation.from_euler("xyz", (0.2, 0.1, -0.3)).apply([0, 0, CF * fc / M_]) - [0, 0, G_]
    np.testing.assert_allclose(sim.get_state()[6:9, 0] * 1e4, want, rtol=1e-10, atol=1e-9)


# ---------------------------------------------------------------------------------- C5: attitude-integral limit
@pytest.mark.parametrize("roll", [0.5, -0.5])
def test_c5_attitude_integral_saturates_exactly_and_torque_stops_growing(cfo, roll):
    """Level, at rest, commanded roll phi held: e_R = (-sin phi, 0, 0) (R_d^T R = Rx(-phi); vee of its skew part), so
    i_R,x = -k sin(phi) h_att until it reaches the limit -+ i_R,max = 0.2 after ceil(0.2 / (|sin phi| h_att)) = 209 ticks,
    then stays exactly there, and tau_x = J_x (k_R sin phi + k_I i_R,max sign(phi)) no longer changes."""
    p = cfo.make_params(0, dict(f_phys=1000.0, f_att=500.0))
    h_att, s = 0.002, math.sin(roll)
    assert abs(p.iR_max - 0.2) < 1e-7 and p.kI[0] > 0
    n_sat = math.ceil(p.iR_max / (abs(s) * h_att))
    assert n_sat == 209
    iR = np.zeros(3)
    taus = []
    for k in range(1, n_sat + 40):
        eR, iR, tau, _ = cfo.attitude_tick(p, [0, 0, 0, 1], [0, 0, 0], [roll, 0, 0, 0.27], iR)
        np.testing.assert_allclose(eR, [-s, 0, 0], atol=1e-16)
        if k < n_sat:
            assert abs(iR[0] + k * s * h_att) < 1e-13 and abs(iR[0]) < p.iR_max
        else:
            assert iR[0] == -math.copysign(p.iR_max, roll)         # exactly the limit, with the sign of the error
        assert iR[1] == 0 and iR[2] == 0
        np.testing.assert_allclose(tau[0], p.J[0] * (p.kR[0] * s - p.kI[0] * iR[0]), rtol=1e-12)
        taus.append(tau[0])
    assert len(set(taus[n_sat - 1:])) == 1 and abs(taus[n_sat - 1]) > abs(taus[n_sat - 3])


def test_c5_integral_limit_inside_the_step_loop(cfo):
    """The same through cfo_step: rotor commands pinned (rpm_min = rpm_max = hover speed, so the body never turns and the
    error stays -sin phi); the ctrl planes carry i_R: 416 steps = 208 ticks below the limit, 2 more steps = at the limit."""
    W = 14476.0
    roll = float(np.float32(0.5))
    sim = cfo.OracleSim(1, 1, 0, dict(integrator=1, iface=cfo.IF_ATTITUDE, f_phys=1000.0, f_att=500.0, rpm_min=W, rpm_max=W,
                                      mass=4 * 3.16e-10 * W * W / G_))
    sim.reset(0)
    sim.set_full(state=fp_state(rpm=(W,) * 4), step_counter=0)
    cm = cmd1([roll, 0, 0, 0.27])
    sim.step(cm, 416, cmd_hold=416)
    assert abs(sim.ctrl()[0, 0] + 208 * math.sin(roll) * 0.002) < 1e-12 and abs(sim.ctrl()[0, 0]) < 0.2
    sim.step(cm, 2, cmd_hold=2)
    lim = sim.ctrl()[0, 0]
    assert lim == -cfo.make_params(0).iR_max                                            # exactly the limit (0.2 as float32)
    sim.step(cm, 100, cmd_hold=100)
    assert sim.ctrl()[0, 0] == lim and np.all(sim.ctrl()[1:3, 0] == 0)
    np.testing.assert_allclose(sim.get_state()[3:7, 0], [0, 0, 0, 1], atol=1e-15)       # the body did not turn


# ---------------------------------------------------------------------------------- C9: Box-Muller component order
def test_c9_box_muller_z0_is_the_cosine_z1_the_sine_of_two_pi_u_b(cfo):
    """(z0, z1) = r (cos 2 pi u_b, sin 2 pi u_b), r = sqrt(-2 ln u_a).  The 23-bit midpoint uniforms never hit 1/4 exactly:
    x_b = 2^30 gives u_b = 1/4 + 2^-24, i.e. the angle pi/2 + d with d = 2 pi 2^-24 -- hand-worked: z0 = -r sin d (tiny,
    negative), z1 = r cos d (= r to 7e-14).  A cos / sin swap, a sign flip of the angle or an angle of pi u_b fails."""
    d = 2 * math.pi * 2.0 ** -24
    xa = 0x80000000                                              # u_a = 1/2 + 2^-24
    r = math.sqrt(-2 * math.log(0.5 + 2.0 ** -24))
    assert cfo.uniform(1 << 30) == 0.25 + 2.0 ** -24 and cfo.uniform(xa) == 0.5 + 2.0 ** -24
    z0, z1 = cfo.normal_pair(xa, 1 << 30)                        # angle pi/2 + d
    assert abs(z0 + r * math.sin(d)) < 1e-15 and abs(z1 - r * math.cos(d)) < 1e-15 and z0 < 0 < z1
    z0, z1 = cfo.normal_pair(xa, 3 << 30)                        # u_b = 3/4 + 2^-24: angle 3 pi/2 + d
    assert abs(z0 - r * math.sin(d)) < 1e-15 and abs(z1 + r * math.cos(d)) < 1e-15 and z1 < 0 < z0
    z0, z1 = cfo.normal_pair(xa, 1 << 31)                        # u_b = 1/2 + 2^-24: angle pi + d
    assert abs(z0 + r * math.cos(d)) < 1e-15 and abs(z1 + r * math.sin(d)) < 1e-15
    z0, z1 = cfo.normal_pair(xa, 1 << 29)                        # u_b = 1/8 + 2^-24: first quadrant, near the diagonal
    assert abs(z0 - r * math.cos(math.pi / 4 + d)) < 1e-15 and abs(z1 - r * math.sin(math.pi / 4 + d)) < 1e-15 and z0 < z1
