"""GPU parity: the CUDA path (through the C ABI, via the thin binding) against the float64 oracle, element by
element on the same seeded inputs.  Tolerances are BASELINE.json:north_star's:
  T1 per-step, teacher-forced: |gpu - oracle| <= 1e-4 * max(|oracle|, floor) per state component
  T2 drift: position error <= 1e-3 m after 1000 free-running steps (hover / tracking runs)
  T3 bit-exact: Philox words, step / tick counters, record-slot table
  T4 reset: <= 2e-6 relative
"""
import math

import numpy as np
import pytest

from util import fresh_oracle, split_calls

pytestmark = pytest.mark.gpu

W_HOVER = math.sqrt(0.027 * 9.81 / (4 * 3.16e-10))
MG = 0.027 * 9.81
FLOOR_FP = np.array([1] * 3 + [1] * 4 + [1] * 3 + [1] * 3 + [W_HOVER] * 4, dtype=np.float64)
FLOOR_AB = np.array([1] * 3 + [1] * 3 + [1] * 3 + [1] * 3 + [MG], dtype=np.float64)
# builder's stricter increment check: rate floors per component
RATE_FP = np.array([1] * 3 + [1] * 4 + [9.81] * 3 + [100] * 3 + [1e5] * 4, dtype=np.float64)
RATE_AB = np.array([1] * 3 + [1] * 3 + [9.81] * 3 + [100] * 3 + [MG / 0.03], dtype=np.float64)


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


def fresh_gpu(cf, wl, **extra):
    sim = cf.Sim(wl.M, wl.N, wl.model, dict(wl.params, **extra))
    sim.reset(wl.seed)
    if wl.broadcast_state is not None:
        sim.set_state(wl.broadcast_state.astype(np.float32), broadcast=True)
    return sim


def floors(model):
    return (FLOOR_FP, RATE_FP) if model == 0 else (FLOOR_AB, RATE_AB)


def assert_state_close(g, o, model, rtol=1e-4, what=""):
    fl = floors(model)[0][:, None]
    err = np.abs(g.astype(np.float64) - o) / np.maximum(np.abs(o), fl)
    j, i = np.unravel_index(np.argmax(err), err.shape)
    assert err.max() <= rtol, f"{what}: component {j} drone {i}: gpu {g[j, i]} oracle {o[j, i]} rel {err.max():.3e}"
    return err.max()


SMALL = dict(cfg1=dict(M=3, n_steps=150), cfg2=dict(M=300, n_steps=160), cfg3=dict(M=700, n_steps=60),
             cfg3b=dict(M=500, n_steps=60), cfg4=dict(M=3, N=333, n_steps=60), cfg5=dict(M=300, n_steps=60),
             cfg5e=dict(M=300, n_steps=60))


# ------------------------------------------------------------------------------------------------ T3 Philox
def test_t3_device_philox_bit_exact_uniform_exact_normals_close(cf, cfo):
    sim = cf.Sim(1, 1, 0)
    rng = np.random.default_rng(3)
    ctr = rng.integers(0, 2 ** 32, (4096, 4), dtype=np.uint64).astype(np.uint32)
    ctr[:8] = [[0, 0, 0, 0], [0xFFFFFFFF] * 4, [1, 2, 3, 4], [7, 0, 999, 1], [5, 0, 0, 2], [5, 0, 1, 2], [5, 1, 0, 2], [6, 0, 0, 3]]
    seed = 0x0123456789ABCDEF
    words, uni, nrm = sim.philox_dev(seed, ctr)
    for k in range(0, 4096, 37):
        want = cfo.philox(seed, ctr[k])
        assert np.array_equal(words[k], want), k
        for c in range(4):
            assert float(uni[k, c]) == cfo.uniform(int(want[c]))                  # exact in float32 (R18)
        z = [*cfo.normal_pair(int(want[0]), int(want[1])), *cfo.normal_pair(int(want[2]), int(want[3]))]
        np.testing.assert_allclose(nrm[k], z, rtol=4e-6, atol=4e-6)
    w0, _, _ = sim.philox_dev(0, np.zeros((1, 4), dtype=np.uint32))
    assert [hex(v) for v in w0[0]] == ["0x6627e8d5", "0xe169c58d", "0xbc57ac4c", "0x9b00dbd8"]


# ------------------------------------------------------------------------------------------------ T4 reset
@pytest.mark.parametrize("name", ["cfg2", "cfg3", "cfg4", "cfg5"])
def test_t4_reset_parity(cf, cfo, W, name):
    wl = W.make(name, seed=5, **SMALL[name])
    g, o = fresh_gpu(cf, wl), fresh_oracle(cfo, wl)
    xs, xo = g.get_state().cpu().numpy(), o.get_state()
    fl = floors(wl.model)[0][:, None]
    assert (np.abs(xs - xo) / np.maximum(np.abs(xo), fl)).max() <= 2e-6
    wg, wo = g.world_params().cpu().numpy(), o.world_params()
    np.testing.assert_allclose(wg, wo, rtol=2e-6, atol=0)
    np.testing.assert_allclose(g.ctrl().cpu().numpy(), o.ctrl(), rtol=2e-6, atol=0)
    assert list(g.counters()) == [0, 0, 0, 0]
    if wl.params.get("n_obstacles"):
        assert np.all(np.isinf(g.min_d2().cpu().numpy()))


# ------------------------------------------------------------------------------------------------ T1 teacher-forced
@pytest.mark.parametrize("seed", [1, 3, 20260601])
@pytest.mark.parametrize("name", ["cfg1", "cfg2", "cfg3", "cfg3b", "cfg4", "cfg5", "cfg5e"])
def test_t1_teacher_forced_single_steps(cf, cfo, W, name, seed):
    """At >= 20 sampled steps (including controller-tick and command-change steps): widen the GPU's own float32
    state / controller planes / world parameters / obstacle minima, advance oracle and GPU one step, compare."""
    wl = W.make(name, seed=seed, **SMALL[name])
    g, o = fresh_gpu(cf, wl), fresh_oracle(cfo, wl)
    fl, rate = floors(wl.model)
    h = 1.0 / wl.params["f_phys"]
    n_checked, worst, worst_rate = 0, 0.0, 0.0
    t = 0
    for cm, n, hold in split_calls(wl, [1, 1, 1, 2, 1, 3, 1, 1, 4, 1]):
        # teacher-force the oracle from the GPU's current float32 data
        xg = g.get_state().cpu().numpy().astype(np.float64)
        md = g.min_d2().cpu().numpy().astype(np.float64) if wl.params.get("n_obstacles") else None
        o.set_full(state=xg, ctrl=g.ctrl().cpu().numpy().astype(np.float64),
                   wparam=g.world_params().cpu().numpy().astype(np.float64), mind2=md, step_counter=t)
        g.step(cm, n, cmd_hold=hold)
        o.step(cm, n, cmd_hold=hold)
        t += n
        if n == 1:
            xn, xo = g.get_state().cpu().numpy().astype(np.float64), o.get_state()
            worst = max(worst, assert_state_close(xn, xo, wl.model, 1e-4, f"{name} step {t}"))
            r = np.abs((xn - xg) - (xo - xg)) / h / rate[:, None]
            worst_rate = max(worst_rate, r.max())
            if md is not None:
                dg, do = np.sqrt(g.min_d2().cpu().numpy().astype(np.float64)), np.sqrt(o.min_d2())
                assert (np.abs(dg - do) <= 1e-4 * np.maximum(do, 1.0)).all()        # T1, floor 1 m on the distance
            n_checked += 1
    assert n_checked >= 20
    assert worst_rate <= 2e-3, worst_rate
    assert list(g.counters())[:3] == list(o.counters())[:3]
    print(f"{name}: {n_checked} teacher-forced steps, worst rel err {worst:.2e}, worst rate err {worst_rate:.2e}")


# ------------------------------------------------------------------------------------------------ free-running
@pytest.mark.parametrize("name", ["cfg1", "cfg2", "cfg3", "cfg3b", "cfg4", "cfg5", "cfg5e"])
def test_free_running_records_counters_and_outputs(cf, cfo, W, name):
    """The whole run in ONE fused launch vs the oracle: every recorded state, the final state, counters (bit-exact),
    record table (bit-exact), controller planes, minimum distance."""
    wl = W.make(name, seed=2, **SMALL[name])
    g, o = fresh_gpu(cf, wl), fresh_oracle(cfo, wl)
    rec_every = wl.record_every
    rg = g.step(wl.cmds, wl.n_steps, cmd_hold=wl.cmd_hold, record_every=rec_every)
    ro = o.step(wl.cmds, wl.n_steps, cmd_hold=wl.cmd_hold, record_every=rec_every)
    tol = 2e-4      # a short free run: float32 rounding accumulates over <= 160 steps, still far below 1e-3
    if ro is not None:
        rgn = rg.cpu().numpy()
        assert rgn.shape == ro.shape
        for k in range(ro.shape[0]):
            assert_state_close(rgn[k], ro[k], wl.model, tol, f"{name} record {k}")
    assert_state_close(g.get_state().cpu().numpy(), o.get_state(), wl.model, tol, f"{name} final")
    assert np.array_equal(g.counters(), o.counters())                             # T3
    assert np.array_equal(g.rec_table(), o.rec_table())                           # T3
    assert g.step_counter == wl.n_steps
    co = o.ctrl()
    cerr = np.abs(g.ctrl().cpu().numpy() - co) / (np.abs(co).max(axis=1, keepdims=True) + 1e-3)
    assert cerr.max() <= 5e-4, cerr.max(axis=1)
    if wl.params.get("n_obstacles"):
        np.testing.assert_allclose(g.min_dist().cpu().numpy(), o.min_dist(), rtol=2e-4, atol=2e-4)


def test_t2_drift_hover_config1(cf, cfo, W):
    """configs[0]: 1000 Euler steps, record every step; position drift <= 1e-3 m, in fused AND single-step mode."""
    wl = W.cfg1(seed=20260601)
    o = fresh_oracle(cfo, wl)
    ro = o.step(wl.cmds, 1000, cmd_hold=1000, record_every=1)
    g = fresh_gpu(cf, wl)
    rg = g.step(wl.cmds, 1000, cmd_hold=1000, record_every=1).cpu().numpy()
    drift = np.abs(rg[:, 0:3, 0] - ro[:, 0:3, 0]).max(axis=1)
    assert drift[-1] <= 1e-3 and drift.max() <= 1e-3, drift.max()
    assert_state_close(rg[-1], ro[-1], 0, 1e-3, "cfg1 step 1000")
    g1 = fresh_gpu(cf, wl)                       # interactive mode: 1000 launches of n_steps = 1
    recs = [g1.step(wl.cmds, 1, cmd_hold=1, record_every=1) for _ in range(1000)]
    r1 = np.stack([r.cpu().numpy()[0] for r in recs])
    np.testing.assert_allclose(r1, rg, rtol=1e-6, atol=1e-7)                       # P20: fused == split
    assert list(g1.counters()) == [1000, 500, 0, 1000] == list(g.counters())
    print(f"cfg1 drift after 1000 steps: {drift[-1]:.3e} m (budget 1e-3)")


def test_t2_drift_tracking_config4(cf, cfo, W):
    """configs[3] shape (M=2 worlds): position controller tracking run, 1000 steps, drift <= 1e-3 m."""
    wl = W.cfg4(seed=20260601, M=2, N=200, n_steps=1000)
    g, o = fresh_gpu(cf, wl), fresh_oracle(cfo, wl)
    g.step(wl.cmds, 1000, cmd_hold=1000)
    o.step(wl.cmds, 1000, cmd_hold=1000)
    xg, xo = g.get_state().cpu().numpy(), o.get_state()
    drift = np.abs(xg[0:3] - xo[0:3]).max()
    assert drift <= 1e-3, drift
    tgt = wl.cmds[0, :, :3].T
    assert np.abs(xo[0:3] - tgt).max() < 0.15                                     # it really tracked its targets
    assert list(g.counters()) == list(o.counters()) == [1000, 0, 200, 0]
    print(f"cfg4 tracking drift after 1000 steps: {drift:.3e} m")


@pytest.mark.parametrize("name", ["cfg2", "cfg3", "cfg4", "cfg5"])
def test_p20_fused_equals_split_on_gpu(cf, W, name):
    wl = W.make(name, seed=4, **SMALL[name])
    rec_every = max(wl.record_every, 1)
    a = fresh_gpu(cf, wl)
    ra = a.step(wl.cmds, wl.n_steps, cmd_hold=wl.cmd_hold, record_every=rec_every).cpu().numpy()
    b = fresh_gpu(cf, wl)
    recs = []
    for cm, n, hold in split_calls(wl, [1, 2, 7, 13]):
        r = b.step(cm, n, cmd_hold=hold, record_every=rec_every)
        if r is not None:
            recs.append(r.cpu().numpy())
    rb = np.concatenate(recs)
    fl = floors(wl.model)[0][None, :, None]
    assert (np.abs(ra - rb) / np.maximum(np.abs(ra), fl)).max() <= 1e-6
    assert np.array_equal(a.counters(), b.counters()) and np.array_equal(a.rec_table(), b.rec_table())


def test_world_offset_shards_reproduce_the_full_run(cf, W):
    """worlds [lo, lo+m) with world_offset = lo give exactly that slice of the full run."""
    wl = W.cfg5(seed=9, M=256, n_steps=30)
    full = fresh_gpu(cf, wl)
    full.step(wl.cmds, 30, cmd_hold=30)
    xf = full.get_state().cpu().numpy()
    for rank in range(2):
        lo, m = W.shard_worlds(256, 2, rank)
        sub = cf.Sim(m, 1, wl.model, dict(wl.params, world_offset=lo))
        sub.reset(wl.seed)
        sub.step(wl.cmds[:, lo:lo + m], 30, cmd_hold=30)
        assert np.array_equal(sub.get_state().cpu().numpy(), xf[:, lo:lo + m])


def test_host_buffer_path_equals_device_path(cf, W):
    import torch
    wl = W.cfg2(seed=6, M=200, n_steps=100)
    a, b = fresh_gpu(cf, wl), fresh_gpu(cf, wl)
    ra = a.step(wl.cmds, 100, cmd_hold=wl.cmd_hold, record_every=10).cpu().numpy()
    ch = torch.from_numpy(wl.cmds).pin_memory()
    rb = b.step_host(ch, 100, cmd_hold=wl.cmd_hold, record_every=10).numpy()
    assert np.array_equal(ra, rb)
    assert np.array_equal(a.get_state().cpu().numpy(), b.get_state_host().numpy())
    w3 = W.cfg3(seed=6, M=300, n_steps=20)
    c, d = fresh_gpu(cf, w3), fresh_gpu(cf, w3)
    c.step(w3.cmds, 20)
    d.step_host(torch.from_numpy(w3.cmds).pin_memory(), 20)
    assert np.array_equal(c.min_dist().cpu().numpy(), d.min_dist_host().numpy())


def test_edge_cases_and_status_codes(cf, W):
    import torch
    sim = cf.Sim(5, 1, 0)
    cm = torch.zeros((1, 5, 4), device="cuda")
    with pytest.raises(cf.CfError) as e:
        sim.step(cm, 1)
    assert e.value.code == cf.E_STATE
    sim.reset(1)
    with pytest.raises(cf.CfError) as e:
        sim.step(cm, 3, cmd_hold=2)
    assert e.value.code == cf.E_SHAPE
    small = torch.empty((1, 17, 5), device="cuda")
    with pytest.raises(cf.CfError) as e:
        sim.step(cm, 4, cmd_hold=4, record_every=2, record=small)
    assert e.value.code == cf.E_BUFFER
    assert sim.step(cm, 3, cmd_hold=3, record_every=5) is None and sim.step_counter == 3      # no record due yet
    r = sim.step(cm, 2, cmd_hold=2, record_every=5)                                            # s = 5 -> one record
    assert r.shape == (1, 17, 5) and list(sim.rec_table()[:2]) == [5, 0]
    # ragged sizes around warp / block boundaries and a single drone
    for M in (1, 31, 33, 257):
        wl = W.cfg2(seed=3, M=M, n_steps=20)
        g = fresh_gpu(cf, wl)
        g.step(wl.cmds, 20, cmd_hold=wl.cmd_hold)
        x = g.get_state().cpu().numpy()
        assert np.isfinite(x).all() and np.allclose(np.linalg.norm(x[3:7], axis=0), 1, atol=1e-6)


@pytest.mark.parametrize("name,M,n_slices", [("cfg3", 5000, 8), ("cfg3", 300, 4), ("cfg3b", 4097, 3), ("cfg3", 33000, 16),
                                              ("cfg2", 2500, 2), ("cfg3", 1 << 20, 8)])   # the last: bench.py's e2e call
def test_rollout_host_equals_step_and_copies(cf, W, name, M, n_slices):
    """cf_rollout_host (sliced launches, result copies on a second stream) returns bit-identical final states, minimum
    distances and counters to cf_set_state + cf_step + cf_get_state + cf_get_aux; a second call continues correctly."""
    import torch
    wl = getattr(W, name)(seed=5, M=M, n_steps=30)
    a, b = fresh_gpu(cf, wl), fresh_gpu(cf, wl)
    cm = torch.from_numpy(np.ascontiguousarray(wl.cmds)).pin_memory()
    x0 = None if wl.broadcast_state is None else torch.from_numpy(wl.broadcast_state.astype(np.float32)).pin_memory()
    obst = wl.params.get("n_obstacles", 0) > 0
    st = torch.empty((wl.D, wl.M), dtype=torch.float32).pin_memory()
    md = torch.empty(wl.M, dtype=torch.float32).pin_memory() if obst else None
    for rep in range(2):
        if x0 is not None:
            a.set_state(x0.cuda(), broadcast=True)
        a.step(cm.cuda(), wl.n_steps, cmd_hold=wl.cmd_hold)
        b.rollout_host(cm, wl.n_steps, st, cmd_hold=wl.cmd_hold, x0_host=x0, min_dist_host=md, n_slices=n_slices)
        assert np.array_equal(st.numpy(), a.get_state().cpu().numpy())
        assert np.array_equal(b.get_state().cpu().numpy(), a.get_state().cpu().numpy())
        if obst:
            assert np.array_equal(md.numpy(), a.min_dist().cpu().numpy())
            assert np.array_equal(b.min_dist().cpu().numpy(), a.min_dist().cpu().numpy())
        assert np.array_equal(a.counters(), b.counters()) and a.step_counter == b.step_counter == (rep + 1) * wl.n_steps


@pytest.mark.parametrize("big,n", [(1000.0, 4), (1.0e5, 1)])
@pytest.mark.parametrize("loop", ["flat_noise", "flat_buffer", "held", "position"])
def test_euler_angles_far_outside_the_mufu_range(cf, cfo, W, loop, big, n):
    """The lean abstracted-model step takes sin / cos of the Euler angles from the MUFU unit: behind a range test in the
    held-command loops (accurate sincosf beyond 2 pi), after a branch-free Cody-Waite reduction in the per-step-command
    loop.  Both must be right for ANY angle: worlds with roll / pitch / yaw of up to +-1000 rad (4 steps) and +-1e5 rad (one
    step from exactly representable inputs: an unreduced MUFU argument is off by |a| 2^-23 = 1e-2 rad there, 2.4e-4 m/s
    in the velocity -- above the 1e-4 bar) against the oracle."""
    M = 300
    if loop == "flat_noise":
        wl = W.cfg3(seed=4, M=M, n_steps=n)
    elif loop == "flat_buffer":
        wl = W.cfg3b(seed=4, M=M, n_steps=n)
    elif loop == "held":
        wl = W.cfg3b(seed=4, M=M, n_steps=2)
        wl.cmd_hold, wl.n_steps = 2, n
    else:
        wl = W.cfg4(seed=4, M=3, N=100, n_steps=n)
    g = cf.Sim(wl.M, wl.N, wl.model, wl.params)
    o = cfo.OracleSim(wl.M, wl.N, wl.model, wl.params)
    g.reset(wl.seed), o.reset(wl.seed)
    x = o.get_state().copy()
    rng = np.random.default_rng(7)
    MN = wl.M * wl.N
    scale = np.where(np.arange(MN) % 3 == 0, big, np.where(np.arange(MN) % 3 == 1, 12.0, 0.4))
    x[3:6] = rng.uniform(-1, 1, (3, MN)) * scale
    x[3:6, :4] = [[6.2831853, -6.2831855, 3.1415927, -3.1415925]] * 3            # at the edges of the tested range
    x32 = x.astype(np.float32)
    g.set_state(x32), o.set_state(x32.astype(np.float64))
    g.step(wl.cmds, wl.n_steps, cmd_hold=wl.cmd_hold), o.step(wl.cmds, wl.n_steps, cmd_hold=wl.cmd_hold)
    assert_state_close(g.get_state().cpu().numpy(), o.get_state(), wl.model, 1e-4, f"large angles, {loop}")
    assert np.array_equal(g.counters(), o.counters())


@pytest.mark.parametrize("case", ["near_the_bound", "foreign_parameters", "nan_state"])
def test_held_command_runs_choose_the_right_loop_body(cf, cfo, W, case):
    """Held-command runs of the abstracted model take the sin / cos test once per run from a bound on the angle growth
    (create-time bounds on the coefficients).  Worlds that start just inside / outside the range with rates that carry
    them across it within the run, parameter planes replaced through cf_set_full (the create-time bounds no longer hold:
    coefficients three times larger), and a NaN state all have to come out as the oracle says."""
    M = 257
    wl = W.cfg3b(seed=6, M=M, n_steps=3)
    wl.cmd_hold, wl.n_steps = 10, 30
    g = cf.Sim(wl.M, 1, wl.model, wl.params)
    o = cfo.OracleSim(wl.M, 1, wl.model, wl.params)
    g.reset(wl.seed), o.reset(wl.seed)
    x = o.get_state().copy()
    rng = np.random.default_rng(3)
    if case == "foreign_parameters":
        wp = o.world_params().copy()
        wp[1:10] *= 3.0                                              # a, b, c of Eq. (10)
        g.set_full(wparam=wp.astype(np.float32)), o.set_full(wparam=wp.astype(np.float32).astype(np.float64))
        x[3:6] = rng.uniform(-3.0, 3.0, (3, M))
        x[9:12] = rng.uniform(-40.0, 40.0, (3, M))
    else:
        x[3:6] = rng.uniform(5.9, 6.6, (3, M)) * rng.choice([-1.0, 1.0], (3, M))
        x[9:12] = rng.uniform(-60.0, 60.0, (3, M))
    if case == "nan_state":
        x[4, ::7] = np.nan
    x32 = x.astype(np.float32)
    g.set_state(x32), o.set_state(x32.astype(np.float64))
    g.step(wl.cmds, wl.n_steps, cmd_hold=wl.cmd_hold), o.step(wl.cmds, wl.n_steps, cmd_hold=wl.cmd_hold)
    xg, xo = g.get_state().cpu().numpy(), o.get_state()
    ok = np.isfinite(xo).all(axis=0)
    assert np.array_equal(ok, np.isfinite(xg).all(axis=0)) and (case != "nan_state" or (~ok).sum() >= M // 7)
    assert_state_close(xg[:, ok], xo[:, ok], wl.model, 2e-4, case)


def test_pair_written_loops_are_selected_and_equal_the_plain_ones(cf, cfo, W):
    """First-principles attitude kernels, tick period 2: calls of an even number of steps from an even step take the
    pair-written loop (REC_*_P / REC_PAIR), everything else the plain one; both give the same trajectory (the oracle's)."""
    for name, rec_every, label in (("cfg2", 10, "REC_TMA_P"), ("cfg2", 0, "REC_NONE_P"), ("cfg1", 1, "REC_SCALAR_P"),
                                   ("cfg2", 1, "REC_PAIR"), ("cfg2", 3, "REC_TMA>")):
        wl = W.make(name, seed=2, **(dict(M=64, n_steps=100) if name == "cfg2" else dict(n_steps=100)))
        g, b, o = fresh_gpu(cf, wl), fresh_gpu(cf, wl), fresh_oracle(cfo, wl)
        rg = g.step(wl.cmds, 100, cmd_hold=wl.cmd_hold, record_every=rec_every)
        assert label in g.describe_launch()[0], (name, rec_every, g.describe_launch()[0])
        ro = o.step(wl.cmds, 100, cmd_hold=wl.cmd_hold, record_every=rec_every)
        recs = []
        for cm, n, hold in split_calls(wl, [7, 20, 33, 40]):                  # odd starts / lengths: the plain loops
            r = b.step(cm, n, cmd_hold=hold, record_every=rec_every)
            assert "_P" not in b.describe_launch()[0] or (n % 2 == 0 and (b.step_counter - n) % 2 == 0)
            if r is not None:
                recs.append(r.cpu().numpy())
        assert_state_close(g.get_state().cpu().numpy(), o.get_state(), wl.model, 2e-4, f"{name} paired")
        fl = floors(wl.model)[0][:, None]
        assert (np.abs(b.get_state().cpu().numpy() - g.get_state().cpu().numpy()) / np.maximum(np.abs(o.get_state()), fl)).max() <= 1e-6
        if rec_every:
            rb = np.concatenate(recs)
            assert rb.shape == tuple(rg.shape) == ro.shape
            assert (np.abs(rb - rg.cpu().numpy()) / np.maximum(np.abs(ro), fl[None])).max() <= 1e-6
        assert np.array_equal(g.counters(), o.counters()) and np.array_equal(b.counters(), o.counters())


def test_rollout_host_status_codes(cf, W):
    import torch
    wl = W.cfg2(seed=1, M=64, n_steps=10)                       # no obstacles: there is no minimum distance to return
    sim = cf.Sim(wl.M, 1, wl.model, wl.params)
    cm = torch.from_numpy(np.ascontiguousarray(wl.cmds)).pin_memory()
    st = torch.empty((wl.D, wl.M), dtype=torch.float32).pin_memory()
    md = torch.empty(wl.M, dtype=torch.float32).pin_memory()
    with pytest.raises(cf.CfError) as e:
        sim.rollout_host(cm, 10, st, cmd_hold=wl.cmd_hold)
    assert e.value.code == cf.E_STATE                           # before cf_reset
    sim.reset(1)
    with pytest.raises(cf.CfError) as e:
        sim.rollout_host(cm, 10, st, cmd_hold=wl.cmd_hold, min_dist_host=md)
    assert e.value.code == cf.E_UNSUPPORTED
    for bad in (0, 17):
        with pytest.raises(cf.CfError) as e:
            sim.rollout_host(cm, 10, st, cmd_hold=wl.cmd_hold, n_slices=bad)
        assert e.value.code == cf.E_ARG
    assert sim.step_counter == 0                                # nothing ran


def test_general_kernel_fidelity_switches(cf, cfo, W):
    """The OPT_ALL instantiations: full Eq. (6), thrust/torque polynomials, Eq. (5) gyro, body drag, all four
    interfaces, RK4 on the abstracted model, simplified AB variant -- teacher-free short runs vs the oracle."""
    base = W.cfg2(seed=8, M=64, n_steps=40)
    extras = dict(cv_up=40.0, cv_dn=25.0, cd_up=2e-4, cd_dn=5e-4, Jp=2.0e-8, Ca=[-0.004, -0.004, -0.002],
                  kf=[1e-3, 2e-7, 3.0e-10], km=[1e-5, 1e-9, 7.9e-12])
    rng = np.random.default_rng(0)
    cases = []
    for integ in (0, 1):
        cases.append((0, dict(base.params, integrator=integ, **extras), base.cmds))
        rot = np.zeros((1, 64, 4), dtype=np.float32) + rng.uniform(12000, 17000, (1, 64, 4)).astype(np.float32)
        cases.append((0, dict(base.params, integrator=integ, iface=0, **extras), rot))
        tq = np.zeros((1, 64, 4), dtype=np.float32)
        tq[..., :3] = rng.uniform(-2e-4, 2e-4, (1, 64, 3))
        tq[..., 3] = 0.3
        cases.append((0, dict(base.params, integrator=integ, iface=1, **extras), tq))
        pos = np.zeros((1, 64, 4), dtype=np.float32)
        pos[..., :3] = rng.uniform(-1, 1, (1, 64, 3)) + [0, 0, 1]
        pos[..., 3] = rng.uniform(-0.5, 0.5, (1, 64))
        cases.append((0, dict(base.params, integrator=integ, iface=3, **extras), pos))
        ab = dict(integrator=integ, f_phys=500.0, init_mode=1, p0_lo=[-1, -1, 0], p0_hi=[1, 1, 2], tilt0_max=0.4,
                  Ca=[-0.004, -0.004, -0.002], dist_sigma=0.003)
        cases.append((1, dict(ab, iface=2), base.cmds))
        cases.append((1, dict(ab, iface=3, ab_thrust_dyn=0), pos))
    for model, prm, cmds in cases:
        hold = 50 if cmds.shape[0] > 1 else 40
        g = cf.Sim(64, 1, model, prm)
        o = cfo.OracleSim(64, 1, model, prm)
        g.reset(8), o.reset(8)
        rg = g.step(cmds, 40, cmd_hold=hold, record_every=8).cpu().numpy()
        ro = o.step(cmds, 40, cmd_hold=hold, record_every=8)
        for k in range(5):
            assert_state_close(rg[k], ro[k], model, 3e-4, f"model {model} iface {prm.get('iface')} integ {prm['integrator']} rec {k}")
        assert np.array_equal(g.counters(), o.counters())


def test_general_kernel_at_sizes_where_the_lean_kernels_take_large_blocks(cf, cfo, W):
    """Requests WITHOUT fidelity extras that have no lean instantiation (position / rotor interface of the first-principles
    model, a randomised nominal plant, RK4 on the abstracted model) run the general kernel, whose launch bound is 128
    threads: with every step recorded at >= 32768 drones the launcher must not hand it the 256 / 512-thread blocks, grouped
    stores or pair-written record modes of the lean record-heavy kernels (decided from the dispatched kernel)."""
    base = W.cfg2(seed=9, M=64, n_steps=6)
    rng = np.random.default_rng(3)
    M = 65536
    pos = np.zeros((1, M, 4), dtype=np.float32)
    pos[..., :3] = rng.uniform(-1, 1, (1, M, 3)) + [0, 0, 1]
    pos[..., 3] = rng.uniform(-0.5, 0.5, (1, M))
    rot = rng.uniform(12000, 17000, (1, M, 4)).astype(np.float32)
    att = np.zeros((1, M, 4), dtype=np.float32)
    att[..., :2] = rng.uniform(-0.2, 0.2, (1, M, 2))
    att[..., 3] = 0.3
    lo, hi = [1.0] * 12, [1.0] * 12
    lo[0], hi[0], lo[4], hi[4] = 0.9, 1.1, 0.95, 1.05
    tq = np.zeros((1, M, 4), dtype=np.float32)
    tq[..., :3] = rng.uniform(-2e-4, 2e-4, (1, M, 3))
    tq[..., 3] = 0.3
    cases = [(0, dict(base.params, iface=3, rnd_lo=lo, rnd_hi=hi), pos), (0, dict(base.params, iface=1, integrator=0), tq),
             (0, dict(base.params, rnd_lo=lo, rnd_hi=hi), att),                     # OPT_RANDP only: was REC_TMA_P on the general kernel
             (1, dict(integrator=1, f_phys=500.0, init_mode=1, p0_lo=[-1, -1, 0], p0_hi=[1, 1, 2], tilt0_max=0.4, iface=2), att)]
    for model, prm, cmds in cases:
        g = cf.Sim(M, 1, model, prm)
        o = cfo.OracleSim(M, 1, model, prm)
        g.reset(9), o.reset(9)
        rg = g.step(cmds, 6, cmd_hold=6, record_every=1).cpu().numpy()
        name, grid, block = g.describe_launch()
        assert "OPT_ALL" in name and block <= 128, (name, block)
        ro = o.step(cmds, 6, cmd_hold=6, record_every=1)
        assert rg.shape == ro.shape == (6, g.D, M)
        for k in (0, 5):
            assert_state_close(rg[k], ro[k], model, 1e-4, f"{name} rec {k}")
        assert np.array_equal(g.counters(), o.counters())
        assert_state_close(g.get_state().cpu().numpy(), o.get_state(), model, 1e-4, name)


@pytest.mark.parametrize("iface,integ", [(0, 0), (0, 1), (3, 0), (3, 1)])
def test_lean_rotor_and_position_interface_kernels_of_the_first_principles_model(cf, cfo, W, iface, integ, monkeypatch):
    """Round 3: compile-time-selected kernels for motor-level control and for the full onboard stack
     on the nominal plant.  Free-running vs the oracle with records in every mode (none / scalar / TMA,
    ragged and aligned sizes, large blocks), and against the general kernel forced by CF_FORCE_GENERAL=1."""
    base = W.cfg2(seed=10, M=64, n_steps=6)
    rng = np.random.default_rng(5)
    for M, n, rec in ((32768, 12, 1), (257, 60, 7), (1024, 40, 0)):
        if iface == 0:
            cmds = rng.uniform(12000, 17000, (2, M, 4)).astype(np.float32)
        else:
            cmds = np.zeros((2, M, 4), dtype=np.float32)
            cmds[..., :3] = rng.uniform(-1, 1, (2, M, 3)) + [0, 0, 1]
            cmds[..., 3] = rng.uniform(-0.5, 0.5, (2, M))
        prm = dict(base.params, iface=iface, integrator=integ, f_pos=100.0)
        hold = -(-n // 2)
        g, o = cf.Sim(M, 1, 0, prm), cfo.OracleSim(M, 1, 0, prm)
        g.reset(10), o.reset(10)
        rg = g.step(cmds, n, cmd_hold=hold, record_every=rec)
        name, _, block = g.describe_launch()
        assert "OPT_ALL" not in name, name
        ro = o.step(cmds, n, cmd_hold=hold, record_every=rec)
        if rec:
            rgn = rg.cpu().numpy()
            assert rgn.shape == ro.shape
            for k in range(ro.shape[0]):
                assert_state_close(rgn[k], ro[k], 0, 2e-4, f"{name} M {M} record {k}")
        assert_state_close(g.get_state().cpu().numpy(), o.get_state(), 0, 2e-4, f"{name} M {M}")
        assert np.array_equal(g.counters(), o.counters()) and np.array_equal(g.rec_table(), o.rec_table())
        co = o.ctrl()
        assert (np.abs(g.ctrl().cpu().numpy() - co) / (np.abs(co).max(axis=1, keepdims=True) + 1e-3)).max() <= 5e-4
        monkeypatch.setenv("CF_FORCE_GENERAL", "1")
        gg = cf.Sim(M, 1, 0, prm)
        monkeypatch.delenv("CF_FORCE_GENERAL")
        gg.reset(10)
        gg.step(cmds, n, cmd_hold=hold, record_every=rec)
        assert "OPT_ALL" in gg.describe_launch()[0]
        assert_state_close(gg.get_state().cpu().numpy(), g.get_state().cpu().numpy().astype(np.float64), 0, 2e-5, "lean vs general")


def test_captured_graph_of_odd_length_never_replays_a_pair_written_kernel(cf, W):
    """A graph [2 steps, 1 step] replayed 4 times starts its 2-step launch at steps 0, 3, 6, 9: the pair-written kernels
    assume an even start, so a call made during stream capture must take the run-time-scheduled kernel."""
    import torch
    wl = W.cfg2(seed=6, M=256, n_steps=12)
    a = fresh_gpu(cf, wl)
    a.step(wl.cmds, 12, cmd_hold=12)
    b = fresh_gpu(cf, wl)
    cm = torch.from_numpy(wl.cmds).cuda()
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        b.bind_stream(side)
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=side):
            b.step(cm, 2, cmd_hold=2)
            assert "_P" not in b.describe_launch()[0] and "REC_PAIR" not in b.describe_launch()[0]
            b.step(cm, 1, cmd_hold=1)
    torch.cuda.current_stream().wait_stream(side)
    for _ in range(4):
        graph.replay()
    torch.cuda.synchronize()
    b.bind_stream()
    b.sync_counters()
    assert b.step_counter == 12 and list(b.counters()) == list(a.counters())
    np.testing.assert_allclose(b.get_state().cpu().numpy(), a.get_state().cpu().numpy(), rtol=1e-6, atol=1e-7)
    c = fresh_gpu(cf, wl)                                  # outside capture the same call does take the pair-written kernel
    c.step(cm, 2, cmd_hold=2)
    assert "_P" in c.describe_launch()[0]


# ------------------------------------------------------------------------------------------------ full BASELINE sizes
def _oracle_slice(cfo, wl, w0, m):
    """The oracle on worlds [w0, w0+m) of the full workload (Philox is keyed by the global world index)."""
    sim = cfo.OracleSim(m, wl.N, wl.model, dict(wl.params, world_offset=w0))
    sim.reset(wl.seed)
    if wl.broadcast_state is not None:
        sim.set_state(wl.broadcast_state, broadcast=True)
    cm = wl.cmds if wl.cmds.ndim == 2 else wl.cmds[:, w0 * wl.N:(w0 + m) * wl.N]
    rec = sim.step(cm, wl.n_steps, cmd_hold=wl.cmd_hold, record_every=wl.record_every)
    return sim, rec


@pytest.mark.parametrize("name", ["cfg2", "cfg3", "cfg4", "cfg5", "cfg5e"])
def test_full_size_sampled_worlds_match_oracle(cf, cfo, W, name):
    """BASELINE.json's full sizes in the launch configuration bench.py times (same Sim, same fused cf_step call, same
    record buffer); sampled worlds are recomputed one slice at a time by the oracle.  Free-running over the full
    horizon, so the bound is the drift budget (1e-3 m on position; 2e-3 relative to the floors on the rest) -- the
    per-step bar is tested teacher-forced above."""
    import torch
    wl = W.make(name)
    g = fresh_gpu(cf, wl)
    rg = g.step(wl.cmds, wl.n_steps, cmd_hold=wl.cmd_hold, record_every=wl.record_every)
    xg = g.get_state().cpu().numpy()
    assert np.isfinite(xg).all()
    md = g.min_dist().cpu().numpy() if wl.params.get("n_obstacles") else None
    m = {"cfg4": 1}.get(name, 16)
    samples = [0, wl.M // 3, wl.M - m]
    rec_slots = None if rg is None else sorted({0, rg.shape[0] // 2, rg.shape[0] - 1})
    for w0 in samples:
        o, ro = _oracle_slice(cfo, wl, w0, m)
        sl = slice(w0 * wl.N, (w0 + m) * wl.N)
        xo = o.get_state()
        assert np.abs(xg[0:3, sl] - xo[0:3]).max() <= 1e-3, (name, w0)
        assert_state_close(xg[:, sl], xo, wl.model, 2e-3, f"{name} world {w0} final")
        if ro is not None:
            for k in rec_slots:
                rk = rg[k, :, sl].cpu().numpy()
                assert np.abs(rk[0:3] - ro[k, 0:3]).max() <= 1e-3
                assert_state_close(rk, ro[k], wl.model, 2e-3, f"{name} world {w0} record {k}")
        if md is not None:
            np.testing.assert_allclose(md[w0:w0 + m], o.min_dist(), rtol=0, atol=1e-3)
    want_att = wl.n_steps // 2 if wl.model == 0 else 0
    want_pos = wl.n_steps // 5 if wl.params.get("iface") == 3 else 0
    assert list(g.counters()) == [wl.n_steps, want_att, want_pos, wl.n_records()]
    del rg, g
    torch.cuda.empty_cache()


def test_cuda_graph_single_step_replay(cf, cfo, W):
    """Interactive mode: ONE captured single-step launch replayed 200 times advances the device-side step counter,
    controller phases and record slots exactly like 200 cf_step(1) calls."""
    import torch
    wl = W.cfg1(seed=5, M=64, n_steps=200)
    a = fresh_gpu(cf, wl)
    a.step(wl.cmds, 200, cmd_hold=200)
    b = fresh_gpu(cf, wl)
    cm = torch.from_numpy(wl.cmds).cuda()
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        b.bind_stream(side)
        b.step(cm, 1, cmd_hold=1)                      # warm-up launch on the capture stream (s = 1)
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=side):
            b.step(cm, 1, cmd_hold=1)                  # captured, not executed
    torch.cuda.current_stream().wait_stream(side)
    for _ in range(199):
        graph.replay()
    torch.cuda.synchronize()
    b.bind_stream()
    b.sync_counters()
    assert b.step_counter == 200
    assert list(b.counters()) == list(a.counters()) == [200, 100, 0, 0]
    np.testing.assert_allclose(b.get_state().cpu().numpy(), a.get_state().cpu().numpy(), rtol=1e-6, atol=1e-7)


def test_lazy_broadcast_reset_and_fused_min_distance(cf, cfo, W):
    """cf_set_state(broadcast) is folded into the next cf_step and the N = 1 minimum distance comes from the rollout
    epilogue; both must be indistinguishable from the eager path and from the oracle."""
    wl = W.cfg3(seed=11, M=777, n_steps=25)
    a = fresh_gpu(cf, wl)                        # reset + set_state(broadcast): pending
    xa = a.get_state().cpu().numpy()             # materialises the pending broadcast
    assert np.array_equal(xa, np.tile(wl.broadcast_state.astype(np.float32)[:, None], (1, 777)))
    assert np.all(np.isinf(a.min_d2().cpu().numpy())) and np.all(a.ctrl().cpu().numpy()[:9] == 0)
    a.step(wl.cmds, 25)                          # eager: planes were written, kernel reads them
    b = fresh_gpu(cf, wl)
    b.step(wl.cmds, 25)                          # lazy: kernel starts from the broadcast vector
    assert np.array_equal(a.get_state().cpu().numpy(), b.get_state().cpu().numpy())
    assert np.array_equal(a.min_d2().cpu().numpy(), b.min_d2().cpu().numpy())
    o = fresh_oracle(cfo, wl)
    o.step(wl.cmds, 25)
    fused = b.min_dist().cpu().numpy()           # epilogue plane
    np.testing.assert_allclose(fused, o.min_dist(), rtol=0, atol=1e-4)
    b.set_full(min_d2=b.min_d2())                # invalidates the epilogue plane -> read-out kernel path
    np.testing.assert_allclose(b.min_dist().cpu().numpy(), fused, rtol=1e-6, atol=1e-7)
    # a second planning iteration: broadcast again, fresh noise (global step counter moved on)
    b.set_state(wl.broadcast_state.astype(np.float32), broadcast=True)
    o.set_state(wl.broadcast_state, broadcast=True)
    b.step(wl.cmds, 25)
    o.step(wl.cmds, 25)
    assert_state_close(b.get_state().cpu().numpy(), o.get_state(), wl.model, 2e-4, "second iteration")
    np.testing.assert_allclose(b.min_dist().cpu().numpy(), o.min_dist(), rtol=0, atol=1e-4)
    assert list(b.counters()) == list(o.counters())


def test_masked_reset_matches_the_oracle(cf, cfo):
    lo, hi = [1.0] * 12, [1.0] * 12
    lo[0], hi[0] = 0.9, 1.1
    ov = dict(integrator=1, iface=2, f_phys=1000.0, f_att=500.0, init_mode=1, p0_lo=[-1, -1, 0], p0_hi=[1, 1, 2],
              tilt0_max=0.5, rnd_lo=lo, rnd_hi=hi, dist_sigma=0.004)
    M, N = 70, 3
    g, o = cf.Sim(M, N, 0, ov), cfo.OracleSim(M, N, 0, ov)
    g.reset(7), o.reset(7)
    cm = np.zeros((1, M * N, 4), dtype=np.float32); cm[..., 0] = 0.1; cm[..., 3] = 0.27
    g.step(cm, 25, cmd_hold=25), o.step(cm, 25, cmd_hold=25)
    mask = (np.random.default_rng(0).random(M) < 0.4).astype(np.uint8)
    before = g.get_state().cpu().numpy()
    g.reset_masked(mask, 99), o.reset_masked(mask, 99)
    x, dm = g.get_state().cpu().numpy(), np.repeat(mask.astype(bool), N)
    assert np.array_equal(x[:, ~dm], before[:, ~dm])                       # untouched worlds: bit-identical
    assert_state_close(x[:, dm], o.get_state()[:, dm], 0, rtol=2e-6, what="masked reset (T4)")
    assert_state_close(x[:, ~dm], o.get_state()[:, ~dm], 0, what="worlds that kept running")
    assert np.abs(g.ctrl().cpu().numpy() - o.ctrl()).max() <= 1e-6 * W_HOVER
    assert np.array_equal(g.counters(), o.counters()) and g.step_counter == 25
    g.step(cm, 30, cmd_hold=30), o.step(cm, 30, cmd_hold=30)
    assert_state_close(g.get_state().cpu().numpy(), o.get_state(), 0, what="after a masked reset")


@pytest.mark.parametrize("name", ["cfg3", "mppi"])
def test_full_size_every_world_against_the_oracle(cf, cfo, W, name):
    """The two planning workloads at their full bench sizes (2^20 x 100 and 500 000 x 250 drone-steps), in the bench's
    launch configuration, with EVERY world compared: the oracle simulates the whole batch (~1 s on the host cores)."""
    wl = W.make(name)
    g, o = fresh_gpu(cf, wl), fresh_oracle(cfo, wl)
    g.step(wl.cmds, wl.n_steps, cmd_hold=wl.cmd_hold)
    o.step(wl.cmds, wl.n_steps, cmd_hold=wl.cmd_hold)
    worst = assert_state_close(g.get_state().cpu().numpy(), o.get_state(), wl.model, 1e-4, f"{name} full size")
    md_g, md_o = g.min_dist().cpu().numpy(), o.min_dist()
    assert np.abs(md_g - md_o).max() <= 1e-4 * max(1.0, np.abs(md_o).max())
    assert np.array_equal(g.counters(), o.counters())
    if name == "mppi":
        Jg, Jo = g.cost().cpu().numpy().astype(np.float64), o.cost()
        assert (np.abs(Jg - Jo) / np.maximum(np.abs(Jo), 1.0)).max() <= 1e-4
    print(f"{name}: {wl.M} worlds x {wl.n_steps} steps, worst relative state error {worst:.2e}")


@pytest.mark.parametrize("name", ["cfg5", "cfg5e"])
def test_full_size_record_mode_every_world_every_100th_record(cf, cfo, W, name):
    """configs[4] at full size in the bench's launch configuration (65 536 worlds x 1000 steps, record every step,
    4.46 GB): every world compared at every 100th recorded step and at the end (T2: position drift <= 1e-3 m)."""
    import torch
    wl = W.make(name)
    g, o = fresh_gpu(cf, wl), fresh_oracle(cfo, wl)
    rg = g.step(wl.cmds, wl.n_steps, cmd_hold=wl.cmd_hold, record_every=1)
    ro = o.step(wl.cmds, wl.n_steps, cmd_hold=wl.cmd_hold, record_every=100)
    assert rg.shape[0] == 1000 and ro.shape[0] == 10
    for k in range(10):
        rk = rg[100 * k + 99].cpu().numpy()
        assert np.abs(rk[0:3] - ro[k, 0:3]).max() <= 1e-3, (name, k)
        assert_state_close(rk, ro[k], wl.model, 2e-3, f"{name} record {100 * k + 99}")
    assert np.array_equal(rg[999].cpu().numpy(), g.get_state().cpu().numpy())          # last record = final state
    assert list(g.counters()) == [1000, 500, 0, 1000]
    del rg
    torch.cuda.empty_cache()


def test_full_size_cfg2_every_world_every_record(cf, cfo, W):
    """configs[1] at full size (4096 worlds x 2000 RK4 steps, 40 command segments, every 10th state recorded): all 200
    records of all worlds against the oracle (T2-style bounds: 1e-3 m on positions, 2e-3 on the other components)."""
    wl = W.make("cfg2")
    g, o = fresh_gpu(cf, wl), fresh_oracle(cfo, wl)
    rg = g.step(wl.cmds, wl.n_steps, cmd_hold=wl.cmd_hold, record_every=wl.record_every).cpu().numpy()
    ro = o.step(wl.cmds, wl.n_steps, cmd_hold=wl.cmd_hold, record_every=wl.record_every)
    assert rg.shape == ro.shape == (200, 17, 4096)
    assert np.abs(rg[:, 0:3] - ro[:, 0:3]).max() <= 1e-3
    for k in range(0, 200, 7):
        assert_state_close(rg[k], ro[k], wl.model, 2e-3, f"cfg2 record {k}")
    assert_state_close(g.get_state().cpu().numpy(), o.get_state(), wl.model, 2e-3, "cfg2 final")
    assert np.array_equal(g.counters(), o.counters()) and np.array_equal(g.rec_table(), o.rec_table())


@pytest.mark.parametrize("model,integ,iface", [(1, 0, 3), (0, 0, 3), (1, 1, 2), (0, 1, 0), (0, 0, 1)])
def test_swarms_without_randomisation_on_superset_kernels(cf, cfo, model, integ, iface):
    """N > 1 with NO per-world randomisation and no record: the dispatcher serves these from instantiations that carry
    OPT_RANDP (they stage the parameter rows of the block's worlds in shared memory), so the staging area must be sized
    from the instantiation, not from the request.  Several worlds per block and a ragged tail."""
    M, N, n = 37, 11, 24
    prm = dict(integrator=integ, iface=iface, init_mode=1, p0_lo=[-1, -1, 0.5], p0_hi=[1, 1, 2], tilt0_max=0.3)
    g, o = cf.Sim(M, N, model, prm), cfo.OracleSim(M, N, model, prm)
    g.reset(4), o.reset(4)
    rng = np.random.default_rng(1)
    cm = np.zeros((2, M * N, 4), dtype=np.float32)
    if iface == 3:
        cm[..., :3] = rng.uniform(-1, 1, (2, M * N, 3)) + [0, 0, 1.2]
        cm[..., 3] = rng.uniform(-0.4, 0.4, (2, M * N))
    elif iface == 2:
        cm[..., :2] = rng.uniform(-0.3, 0.3, (2, M * N, 2)); cm[..., 3] = rng.uniform(0.2, 0.35, (2, M * N))
    elif iface == 1:
        cm[..., :3] = rng.uniform(-2e-4, 2e-4, (2, M * N, 3)); cm[..., 3] = rng.uniform(0.2, 0.35, (2, M * N))
    else:
        cm[...] = rng.uniform(12000, 17000, (2, M * N, 4))
    g.step(cm, n, cmd_hold=12), o.step(cm, n, cmd_hold=12)
    assert_state_close(g.get_state().cpu().numpy(), o.get_state(), model, 2e-4, f"model {model} integ {integ} iface {iface}")
    assert np.array_equal(g.counters(), o.counters())
    g.step(cm, n, cmd_hold=12, record_every=5)          # the same simulator again WITH the tiled-record staging area
    assert np.isfinite(g.get_state().cpu().numpy()).all()


@pytest.mark.parametrize("name,kw,rec_every", [("cfg2", dict(M=256, n_steps=120), 3), ("cfg5", dict(M=96, n_steps=50), 1),
                                               ("cfg5e", dict(M=2048, n_steps=40), 1), ("cfg4", dict(M=2, N=160, n_steps=60), 7),
                                               ("cfg1", dict(M=32, n_steps=33), 1)])
def test_tma_record_path_small_sizes(cf, cfo, W, name, kw, rec_every):
    """Drone counts that are multiples of 32 take the bulk-tensor (TMA) record store: every record of every drone against
    the oracle, in one fused call and in a split run whose calls start at odd record slots (tile double-buffering, row
    coordinate = slot * D of the call's own record buffer), counters and record table bit-exact."""
    wl = W.make(name, seed=12, **kw)
    assert wl.MN % 32 == 0
    g, o = fresh_gpu(cf, wl), fresh_oracle(cfo, wl)
    assert "REC_NONE" in g.describe_launch()[0]
    rg = g.step(wl.cmds, wl.n_steps, cmd_hold=wl.cmd_hold, record_every=rec_every).cpu().numpy()
    # configs[4] proper (RK4, every step recorded, an even run from an even step) takes the pair-scheduled kernel
    assert ("REC_PAIR" if name == "cfg5" else "REC_TMA") in g.describe_launch()[0]
    ro = o.step(wl.cmds, wl.n_steps, cmd_hold=wl.cmd_hold, record_every=rec_every)
    assert rg.shape == ro.shape and rg.shape[0] == wl.n_steps // rec_every
    for k in range(ro.shape[0]):
        assert_state_close(rg[k], ro[k], wl.model, 2e-4, f"{name} record {k}")
    assert np.array_equal(g.counters(), o.counters()) and np.array_equal(g.rec_table(), o.rec_table())
    b = fresh_gpu(cf, wl)
    recs = []
    for cm, n, hold in split_calls(wl, [1, 2, 5, 3, 11]):
        r = b.step(cm, n, cmd_hold=hold, record_every=rec_every)
        assert "REC_PAIR" not in b.describe_launch()[0] or (n % 2 == 0 and (b.step_counter - n) % 2 == 0)
        if r is not None:
            recs.append(r.cpu().numpy())
    rb = np.concatenate(recs)
    fl = floors(wl.model)[0][None, :, None]
    assert rb.shape == rg.shape and (np.abs(rb - rg) / np.maximum(np.abs(rg), fl)).max() <= 1e-6
    assert np.array_equal(b.counters(), g.counters()) and np.array_equal(b.rec_table(), g.rec_table())
