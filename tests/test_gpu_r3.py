"""Round-3 GPU parity cases for what VERDICT r2 found exercised nowhere: Eq. (8)'s thrust scaling c_f != 1 (lean and
general rollout kernels, both adjoint paths), runs that reach the attitude-integral limit of C5 (rollout and adjoint:
reading R33, zero derivative through an active clip), and BASELINE.json configs[3] at full size against the oracle for
EVERY world and record.  Bars as in test_gpu_parity.py / test_gpu_grad.py (north_star: 1e-4 relative per step with the
state floors, 1e-3 m position drift; short free runs 2e-4).  The oracle side of each is pinned in
tests/test_oracle_pins_r3.py.
"""
import numpy as np
import pytest

from test_gpu_parity import _oracle_slice, assert_state_close, fresh_gpu, fresh_oracle

pytestmark = pytest.mark.gpu

GOAL = [0.5, -0.2, 1.2]


@pytest.fixture(scope="module")
def cf():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2606_01478_b200 import build, cf as m
    build.build()
    m.lib()
    return m


@pytest.fixture(scope="module")
def W():
    from paper_2606_01478_b200 import workloads
    return workloads


@pytest.fixture(scope="module")
def og():
    from oracle import grad
    return grad


# ------------------------------------------------------------------------------------------------ Eq. (8): c_f != 1
@pytest.mark.parametrize("name,kw,extra,lean", [
    ("cfg3", dict(M=700, n_steps=60), dict(ab_cf=0.8), True),                       # lean Euler kernel, in-kernel noise
    ("cfg3b", dict(M=500, n_steps=60), dict(ab_cf=1.15), True),                     # lean Euler kernel, command buffer
    ("cfg4", dict(M=3, N=333, n_steps=60), dict(ab_cf=0.85), True),                 # lean position-interface kernel
    ("cfg3b", dict(M=500, n_steps=60), dict(ab_cf=0.8, integrator=1), False),       # general kernel: RK4 on the AB model
    ("cfg3b", dict(M=500, n_steps=60), dict(ab_cf=0.8, ab_thrust_dyn=0), False),    # general kernel: simplified variant
])
def test_thrust_scaling_coefficient_cf_in_the_rollout_kernels(cf, cfo, W, name, kw, extra, lean):
    wl = W.make(name, seed=5, **kw)
    g, o = fresh_gpu(cf, wl, **extra), cfo.OracleSim(wl.M, wl.N, wl.model, dict(wl.params, **extra))
    o.reset(wl.seed)
    if wl.broadcast_state is not None:
        o.set_state(wl.broadcast_state, broadcast=True)
    ref = fresh_oracle(cfo, wl)                                    # the same run with c_f = 1: the coefficient must matter
    rg = g.step(wl.cmds, wl.n_steps, cmd_hold=wl.cmd_hold, record_every=10).cpu().numpy()
    kernel = g.describe_launch()[0]
    assert ("OPT_ALL" not in kernel) == lean, kernel
    ro = o.step(wl.cmds, wl.n_steps, cmd_hold=wl.cmd_hold, record_every=10)
    ref.step(wl.cmds, wl.n_steps, cmd_hold=wl.cmd_hold)
    for k in range(ro.shape[0]):
        assert_state_close(rg[k], ro[k], wl.model, 2e-4, f"{kernel} record {k}")
    assert_state_close(g.get_state().cpu().numpy(), o.get_state(), wl.model, 2e-4, kernel)
    assert np.array_equal(g.counters(), o.counters())
    if "integrator" not in extra and "ab_thrust_dyn" not in extra:
        assert np.abs(o.get_state()[8] - ref.get_state()[8]).max() > 0.05          # v_z differs visibly from the c_f = 1 run
    if wl.params.get("n_obstacles"):
        np.testing.assert_allclose(g.min_dist().cpu().numpy(), o.min_dist(), rtol=2e-4, atol=2e-4)


def _att_cmds(K, M, seed, amp=0.2):
    rng = np.random.default_rng(seed)
    c = np.zeros((K, M, 4), dtype=np.float32)
    c[..., :2] = rng.uniform(-amp, amp, (K, M, 2))
    c[..., 2] = rng.uniform(-0.1, 0.1, (K, M))
    c[..., 3] = rng.uniform(0.2, 0.35, (K, M))
    return c


def _grad_compare(g_gpu, L_gpu, L_o, g_o, tol=1e-3):
    from test_gpu_grad import compare
    return compare(g_gpu, L_gpu, L_o, g_o, tol)


@pytest.mark.parametrize("extra", [dict(integrator=0), dict(integrator=1), dict(integrator=1, dist_sigma=0.004),
                                   dict(integrator=0, iface=3, f_pos=100.0)])
def test_thrust_scaling_coefficient_cf_in_the_adjoint_kernels(cf, cfo, og, extra):
    """cf_grad on the abstracted model with c_f = 0.8: lean adjoint (Euler / RK4, attitude and position interface) and the
    general adjoint (force disturbances).  d v / d f_cmd carries c_f, so dropping it is a 25 % error on the thrust channel."""
    M = 200
    params = dict(dict(iface=2, f_phys=500.0, f_att=500.0, init_mode=1, p0_lo=[-1, -1, 0.5], p0_hi=[1, 1, 2], tilt0_max=0.3,
                       ab_cf=0.8), **extra)
    g, o = cf.Sim(M, 1, 1, params), cfo.OracleSim(M, 1, 1, params)
    g.reset(3), o.reset(3)
    if params["iface"] == 3:
        rng = np.random.default_rng(1)
        cmds = np.zeros((4, M, 4), dtype=np.float32)
        cmds[..., :3] = o.get_state()[:3].T[None] + rng.uniform(-0.3, 0.3, (4, M, 3))
        cmds[..., 3] = rng.uniform(-0.4, 0.4, (4, M))
        hold = 5
    else:
        cmds, hold = _att_cmds(4, M, seed=2, amp=0.3), 5
    L_gpu, g_gpu = g.grad(cmds, 20, GOAL, cmd_hold=hold)
    L_o, g_o = og.value_and_grad(o, cmds, 20, hold, GOAL)
    _grad_compare(g_gpu.cpu().numpy(), L_gpu.cpu().numpy(), L_o, g_o)
    assert np.abs(g_o).max() > 0


# ------------------------------------------------------------------------------------------------ C5: integral limit
SAT = dict(kI=[2000.0, 2000.0, 2000.0], iR_max=2e-3)      # gains that make the integral term matter and saturate in a few ticks


@pytest.mark.parametrize("integrator,extra", [(1, {}), (0, {}), (1, dict(dist_sigma=0.004))])
def test_rollout_that_reaches_the_attitude_integral_limit(cf, cfo, W, integrator, extra):
    """configs[1] recipe with k_I = 2000, i_R,max = 2e-3: every drone crosses the limit (both signs, at different ticks) and
    leaves it again when the error changes sign.  Lean kernels and, with disturbances but no randomisation, the general one."""
    wl = W.cfg2(seed=7, M=300, n_steps=160)
    prm = dict(wl.params, integrator=integrator, **SAT, **extra)
    g, o = cf.Sim(wl.M, 1, 0, prm), cfo.OracleSim(wl.M, 1, 0, prm)
    g.reset(7), o.reset(7)
    rg = g.step(wl.cmds, 160, cmd_hold=wl.cmd_hold, record_every=10).cpu().numpy()
    ro = o.step(wl.cmds, 160, cmd_hold=wl.cmd_hold, record_every=10)
    kernel = g.describe_launch()[0]
    for k in range(16):
        assert_state_close(rg[k], ro[k], 0, 2e-4, f"{kernel} record {k}")
    io, ig = o.ctrl()[0:3], g.ctrl().cpu().numpy()[0:3]
    lim = 2e-3                                  # the oracle holds the parameter as a double, the GPU as float32(2e-3)
    at_limit = np.abs(io) == lim
    assert at_limit[:2].mean() > 0.3 and (io == lim).any() and (io == -lim).any() and (~at_limit).any()
    assert np.array_equal(np.abs(ig) == np.float32(lim), at_limit)                  # the same drones sit on the limit, exactly
    assert np.abs(ig - io).max() <= 1e-4 * lim + 1e-9
    assert np.array_equal(g.counters(), o.counters())


def test_pinned_rotor_run_saturates_at_exactly_the_limit_on_the_gpu(cf, cfo):
    """The closed-form case of tests/test_oracle_pins_r3.py on the GPU: rotors pinned to hover speed, roll command 0.5 held,
    default gains: i_R,x = -k sin(0.5) 0.002 for 208 ticks, then exactly -0.2."""
    Wh, roll = 14476.0, float(np.float32(0.5))
    prm = dict(integrator=1, iface=2, f_phys=1000.0, f_att=500.0, rpm_min=Wh, rpm_max=Wh, mass=4 * 3.16e-10 * Wh * Wh / 9.81)
    g, o = cf.Sim(64, 1, 0, prm), cfo.OracleSim(64, 1, 0, prm)
    g.reset(0), o.reset(0)
    x0 = np.zeros((17, 64)); x0[2] = 1; x0[6] = 1; x0[13:] = Wh
    g.set_full(state=x0.astype(np.float32), step_counter=0), o.set_full(state=x0, step_counter=0)
    cm = np.zeros((1, 64, 4), dtype=np.float32); cm[..., 0] = roll; cm[..., 3] = 0.27
    g.step(cm, 416, cmd_hold=416), o.step(cm, 416, cmd_hold=416)
    ig = g.ctrl().cpu().numpy()[0]
    assert np.abs(ig - o.ctrl()[0]).max() <= 1e-4 * 0.2 and (np.abs(ig) < 0.2).all()
    assert abs(ig[0] + 208 * np.sin(roll) * 0.002) <= 2e-5
    g.step(cm, 2, cmd_hold=2), o.step(cm, 2, cmd_hold=2)
    assert (g.ctrl().cpu().numpy()[0] == -np.float32(0.2)).all() and (o.ctrl()[0] == -cfo.make_params(0).iR_max).all()
    g.step(cm, 100, cmd_hold=100)
    assert (g.ctrl().cpu().numpy()[0] == -np.float32(0.2)).all() and (g.ctrl().cpu().numpy()[1:3] == 0).all()


@pytest.mark.parametrize("integrator,iR_max,extra", [(1, 2e-3, {}), (0, 2e-3, {}), (1, 0.2, {}), (1, 2e-3, dict(dist_sigma=0.004))])
def test_gradient_through_a_saturated_attitude_integral_is_cut(cf, cfo, og, integrator, iR_max, extra):
    """Reading R33 in cf_grad: where the integral clip is active the derivative through i_R is 0.  40 warm-up steps against
    a large held attitude error drive roll / pitch integrals of every drone deep into the limit (i_R,max = 2e-3; the error
    keeps its sign over the differentiated steps, so the central differences of the oracle stay on one branch); with
    k_I = 2000 the integral path is 3 % of the proportional one (k_I h_att / k_R), 30 x the tolerance -- an adjoint that
    ignored the clip fails.  i_R,max = 0.2 is the same run with nobody at the limit (the path is live and must be right)."""
    M = 192
    prm = dict(integrator=integrator, iface=2, f_phys=1000.0, f_att=500.0, init_mode=1, p0_lo=[-1, -1, 0], p0_hi=[1, 1, 2],
               tilt0_max=0.1, kI=SAT["kI"], iR_max=iR_max, **extra)
    g, o = cf.Sim(M, 1, 0, prm), cfo.OracleSim(M, 1, 0, prm)
    g.reset(3), o.reset(3)
    rng = np.random.default_rng(8)
    sign = np.where(rng.random((M, 2)) < 0.5, -1.0, 1.0)
    warm = np.zeros((1, M, 4), dtype=np.float32)
    warm[0, :, :2] = 0.45 * sign
    warm[0, :, 3] = 0.27
    g.step(warm, 40, cmd_hold=40), o.step(warm, 40, cmd_hold=40)
    assert ((np.abs(o.ctrl()[0:2]) == iR_max).all()) == (iR_max < 0.1)        # (the oracle holds the limit as a double)
    assert ((np.abs(g.ctrl().cpu().numpy()[0:2]) == np.float32(iR_max)).all()) == (iR_max < 0.1)
    cmds = np.zeros((6, M, 4), dtype=np.float32)
    cmds[:, :, :2] = (0.45 + rng.uniform(-0.04, 0.04, (6, M, 2))) * sign[None]
    cmds[:, :, 2] = rng.uniform(-0.05, 0.05, (6, M))
    cmds[:, :, 3] = rng.uniform(0.22, 0.32, (6, M))
    L_gpu, g_gpu = g.grad(cmds, 10, GOAL, cmd_hold=2)
    L_o, g_o = og.value_and_grad(o, cmds, 10, 2, GOAL)
    _grad_compare(g_gpu.cpu().numpy(), L_gpu.cpu().numpy(), L_o, g_o)
    assert (g_gpu[5] == 0).all().item() and np.abs(g_o[:5, :, :2]).max() > 0


# ------------------------------------------------------------------------------------------------ configs[3], all of it
def test_full_size_cfg4_every_world_every_record(cf, cfo, W):
    """BASELINE.json configs[3] (1000 worlds x 4000 drones, 500 steps, 10 records) in the launch configuration bench.py
    times, against the oracle for all 4 * 10^6 drones at all 10 records and the final state -- the oracle recomputes the run
    50 worlds at a time.  Free-running over the full horizon: position drift <= 1e-3 m (north_star), the other components
    2e-3 relative to the floors (as in test_full_size_sampled_worlds_match_oracle)."""
    import torch
    wl = W.make("cfg4")
    g = fresh_gpu(cf, wl)
    rg = g.step(wl.cmds, wl.n_steps, cmd_hold=wl.cmd_hold, record_every=wl.record_every)
    assert rg.shape == (10, 13, wl.M * wl.N)
    xg = g.get_state()
    m, worst_p, worst = 50, 0.0, 0.0
    for w0 in range(0, wl.M, m):
        o, ro = _oracle_slice(cfo, wl, w0, m)
        sl = slice(w0 * wl.N, (w0 + m) * wl.N)
        rk = rg[:, :, sl].cpu().numpy()
        worst_p = max(worst_p, np.abs(rk[:, 0:3] - ro[:, 0:3]).max())
        for k in range(10):
            worst = max(worst, assert_state_close(rk[k], ro[k], wl.model, 2e-3, f"cfg4 worlds {w0}.. record {k}"))
        worst = max(worst, assert_state_close(xg[:, sl].cpu().numpy(), o.get_state(), wl.model, 2e-3, f"cfg4 worlds {w0}.. final"))
        assert worst_p <= 1e-3, (w0, worst_p)
    assert list(g.counters()) == [500, 0, 100, 10]
    print(f"cfg4 full size, every world and record: worst position drift {worst_p:.2e} m, worst relative error {worst:.2e}")
    del rg, g
    torch.cuda.empty_cache()


# ------------------------------------------------------------------------------------------------ checkpoint / resume
@pytest.mark.parametrize("name,kw,cut", [("cfg5", dict(M=300, n_steps=60), 23), ("cfg4", dict(M=3, N=333, n_steps=60), 31),
                                         ("cfg3", dict(M=700, n_steps=60), 17)])
def test_checkpoint_at_an_odd_step_restored_into_a_fresh_simulator_continues_bit_for_bit(cf, W, name, kw, cut):
    """SURVEY.md section 5 / cf.h "A COMPLETE CHECKPOINT": run `cut` steps, read everything out, restore into a NEW
    simulator, run the rest; states, records, controller planes, obstacle minima, counters and the record-slot table equal
    those of the uninterrupted run bit for bit (randomised plant + Philox disturbances; position controller with integrals;
    planning rollout with its AR(1) noise state, running cost and obstacle minima)."""
    from util import split_calls
    wl = W.make(name, seed=12, **kw)
    rec = 3
    (cm1, n1, h1), (cm2, n2, h2) = split_calls(wl, [cut, wl.n_steps])      # the same two cf_step calls on both sides
    assert n1 == cut and n1 + n2 == wl.n_steps
    a = fresh_gpu(cf, wl)                                          # uninterrupted: the two calls back to back on one simulator
    ra = np.concatenate([a.step(cm1, n1, cmd_hold=h1, record_every=rec).cpu().numpy(),
                         a.step(cm2, n2, cmd_hold=h2, record_every=rec).cpu().numpy()])
    b = fresh_gpu(cf, wl)
    rb1 = b.step(cm1, n1, cmd_hold=h1, record_every=rec)
    ck = dict(state=b.get_state().clone(), ctrl=b.ctrl(), wparam=b.world_params(), counters=b.counters(), table=b.rec_table(),
              min_d2=b.min_d2() if wl.params.get("n_obstacles") else None,
              eps=b.eps() if wl.params.get("noise_beta") else None, cost_run=b.cost_run() if wl.params.get("cost_on") else None)
    assert ck["counters"][0] == cut
    del b
    c = cf.Sim(wl.M, wl.N, wl.model, wl.params)
    c.reset(wl.seed)                                               # the seed of the disturbance / noise streams
    c.set_full(state=ck["state"], ctrl=ck["ctrl"], wparam=ck["wparam"], min_d2=ck["min_d2"])
    if ck["eps"] is not None or ck["cost_run"] is not None:
        c.set_plan_state(eps=ck["eps"], cost_run=ck["cost_run"])
    c.set_counters(ck["counters"], ck["table"])
    assert c.step_counter == cut and np.array_equal(c.counters(), ck["counters"])
    rc2 = c.step(cm2, n2, cmd_hold=h2, record_every=rec)
    assert np.array_equal(np.concatenate([rb1.cpu().numpy(), rc2.cpu().numpy()]).view(np.uint32), ra.view(np.uint32))
    assert np.array_equal(c.get_state().cpu().numpy().view(np.uint32), a.get_state().cpu().numpy().view(np.uint32))
    assert np.array_equal(c.ctrl().cpu().numpy().view(np.uint32), a.ctrl().cpu().numpy().view(np.uint32))
    assert np.array_equal(c.counters(), a.counters()) and np.array_equal(c.rec_table(), a.rec_table())
    assert c.counters()[3] == wl.n_steps // rec
    if wl.params.get("n_obstacles"):
        assert np.array_equal(c.min_d2().cpu().numpy(), a.min_d2().cpu().numpy())
        assert np.array_equal(c.min_dist().cpu().numpy(), a.min_dist().cpu().numpy())
    if wl.params.get("cost_on"):
        assert np.array_equal(c.cost().cpu().numpy(), a.cost().cpu().numpy())


def test_nonfinite_debug_counter(cf, W):
    wl = W.cfg2(seed=3, M=1000, n_steps=10)
    g = fresh_gpu(cf, wl)
    g.step(wl.cmds, 10, cmd_hold=wl.cmd_hold)
    assert g.nonfinite() == (0, None)
    x = g.get_state().clone()
    x[9, 713] = float("nan"); x[0, 40] = float("inf"); x[16, 999] = float("-inf"); x[3, 40] = float("nan")
    g.set_full(state=x)
    assert g.nonfinite() == (3, 40)


def test_rollout_host_on_a_caller_owned_copy_stream(cf, W):
    """cf_set_copy_stream: the result copies of cf_rollout_host run on the caller's stream; same bits as on the library's."""
    import torch
    wl = W.cfg3(seed=9, M=5000, n_steps=20)
    cm = torch.from_numpy(np.ascontiguousarray(wl.cmds)).pin_memory()
    x0 = torch.from_numpy(wl.broadcast_state.astype(np.float32)).pin_memory()
    outs = []
    mine = torch.cuda.Stream()
    for stream in (None, mine, None):
        sim = cf.Sim(wl.M, 1, wl.model, wl.params)
        sim.reset(wl.seed)
        if stream is not None:
            sim.set_copy_stream(stream)
        st = torch.empty((wl.D, wl.M), dtype=torch.float32).pin_memory()
        md = torch.empty(wl.M, dtype=torch.float32).pin_memory()
        sim.rollout_host(cm, 20, st, cmd_hold=wl.cmd_hold, min_dist_host=md, x0_host=x0, n_slices=4)
        if stream is not None:
            sim.set_copy_stream(None)                              # back to a library-owned stream: created on the next call
            st2 = torch.empty_like(st).pin_memory()
            sim.rollout_host(cm, 20, st2, cmd_hold=wl.cmd_hold, x0_host=x0, n_slices=3)
        outs.append((st.numpy().copy(), md.numpy().copy()))
    for s, m in outs[1:]:
        assert np.array_equal(s, outs[0][0]) and np.array_equal(m, outs[0][1])
