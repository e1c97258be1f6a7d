"""GPU parity of the sampling-based planner (R25-R32) through the C ABI:
planning rollout (AR(1) noise, per-controller nominal, rollout cost) against oracle/cfo.c, and cf_mppi_update /
cf_mppi_iterate against oracle/mppi.py.

Bars: elite index sets, best controller and thresholds are integer / bit-pattern work -> exact, with the selection
taken on the same float32 costs on both sides (the kernel's precision); states, costs, weights and means are floating
point -> the tolerances written below (north_star's 1e-4 per component with the state floors; commands: 5e-6 absolute,
from the 4e-6 bound on the MUFU Box-Muller normals times sigma <= 0.4 plus float32 summation over the elites).
"""
import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

MG = 0.027 * 9.81
FLOOR_AB = np.array([1] * 3 + [1] * 3 + [1] * 3 + [1] * 3 + [MG], dtype=np.float64)[:, None]


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
def mp():
    from oracle import mppi
    return mppi


def pair(cf, cfo, wl, **extra):
    g = cf.Sim(wl.M, 1, wl.model, dict(wl.params, **extra))
    o = cfo.OracleSim(wl.M, 1, wl.model, dict(wl.params, **extra))
    g.reset(wl.seed), o.reset(wl.seed)
    return g, o


def rel_state_err(g, o):
    return (np.abs(g.astype(np.float64) - o) / np.maximum(np.abs(o), FLOOR_AB)).max()


def random_nominal(wl, seed=0, amp=0.2):
    rng = np.random.default_rng(seed)
    nom = wl.cmds.copy()
    nom[..., :2] += rng.uniform(-amp, amp, nom[..., :2].shape).astype(np.float32)
    nom[..., 3] += rng.uniform(-0.03, 0.03, nom[..., 3].shape).astype(np.float32)
    return nom


def oracle_update(mp, wl, cost_f32, nominal, s_start, n_elite=None, lam=None, shift=None):
    p, n = wl.params, wl.notes
    return mp.update(cost_f32, nominal, seed=wl.seed, world_offset=int(p.get("world_offset", 0)),
                     worlds_per_ctrl=p["worlds_per_ctrl"], s_start=s_start, cmd_hold=wl.cmd_hold,
                     sigma=p["noise_sigma"], beta=p["noise_beta"], lo=p["cmd_lo"], hi=p["cmd_hi"],
                     n_elite=n["n_elite"] if n_elite is None else n_elite, lam=n["lam"] if lam is None else lam,
                     shift=n["shift"] if shift is None else shift)


# --------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("lazy", [True, False])
def test_planning_rollout_state_noise_and_cost_match_the_oracle(cf, cfo, W, lazy):
    wl = W.mppi(seed=3, n_ctrl=3, worlds_per_ctrl=211, horizon=6, cmd_hold=5, n_elite=7)     # M = 633: ragged tail
    g, o = pair(cf, cfo, wl)
    nom = random_nominal(wl)
    warm = wl.cmds[:, :1].copy()
    g.step(warm, 3, cmd_hold=3), o.step(warm, 3, cmd_hold=3)       # step counter off zero, noise chain started
    x0 = wl.broadcast_state
    g.set_state(x0.astype(np.float32), broadcast=True), o.set_state(x0, broadcast=True)
    if not lazy:
        g.get_state()                                             # materialises the broadcast: planes are read back
        assert np.isnan(g.eps().cpu().numpy()[0]).all() and (g.cost_run().cpu().numpy() == 0).all()
    g.step(nom, wl.n_steps, cmd_hold=wl.cmd_hold), o.step(nom, wl.n_steps, cmd_hold=wl.cmd_hold)
    assert np.array_equal(g.counters(), o.counters())
    assert rel_state_err(g.get_state().cpu().numpy(), o.get_state()) <= 1e-4
    np.testing.assert_allclose(g.eps().cpu().numpy(), o.eps(), rtol=0, atol=2e-5)
    np.testing.assert_allclose(g.ctrl().cpu().numpy()[6:10], o.ctrl()[6:10], rtol=0, atol=5e-6)   # last applied command
    Jo, Jg = o.cost(), g.cost().cpu().numpy().astype(np.float64)
    assert (np.abs(Jg - Jo) / np.maximum(np.abs(Jo), 1.0)).max() <= 1e-4
    Ro, Rg = o.cost_run(), g.cost_run().cpu().numpy().astype(np.float64)
    assert (np.abs(Rg - Ro) / np.maximum(np.abs(Ro), 1.0)).max() <= 1e-4
    np.testing.assert_allclose(g.min_dist().cpu().numpy(), o.min_dist(), rtol=0, atol=1e-4)
    assert (Jo > Ro).all() and np.ptp(Jo) > 0.01                   # the terminal / obstacle terms are live


def test_planning_rollout_fused_equals_knot_by_knot_and_teacher_forced_step(cf, cfo, W):
    wl = W.mppi(seed=4, n_ctrl=2, worlds_per_ctrl=160, horizon=5, cmd_hold=4, n_elite=5)
    nom = random_nominal(wl, 1)
    g, o = pair(cf, cfo, wl)
    g2, _ = pair(cf, cfo, wl)
    x0 = wl.broadcast_state.astype(np.float32)
    g.set_state(x0, broadcast=True), g2.set_state(x0, broadcast=True)
    g.step(nom, wl.n_steps, cmd_hold=wl.cmd_hold)
    for t in range(5):
        g2.step(nom[:, t:t + 1].copy(), 4, cmd_hold=4)             # eps / cost planes round-trip through HBM
        if t == 2:                                                 # teacher-forced: oracle continues from the GPU's planes
            o.set_full(state=g2.get_state().cpu().numpy(), ctrl=g2.ctrl().cpu().numpy(),
                       wparam=g2.world_params().cpu().numpy(), mind2=g2.min_d2().cpu().numpy(), step_counter=12)
            o.set_plan_state(eps=g2.eps().cpu().numpy(), cost_run=g2.cost_run().cpu().numpy())
    o.step(nom[:, 3:].copy(), 8, cmd_hold=4)
    a, b = g.get_state().cpu().numpy(), g2.get_state().cpu().numpy()
    assert np.abs(a - b).max() <= 1e-6
    np.testing.assert_allclose(g.cost().cpu().numpy(), g2.cost().cpu().numpy(), rtol=2e-6)
    np.testing.assert_allclose(g.eps().cpu().numpy(), g2.eps().cpu().numpy(), rtol=0, atol=1e-6)
    assert rel_state_err(b, o.get_state()) <= 1e-4
    np.testing.assert_allclose(g2.eps().cpu().numpy(), o.eps(), rtol=0, atol=1e-5)
    Jo = o.cost()
    assert (np.abs(g2.cost().cpu().numpy() - Jo) / np.maximum(np.abs(Jo), 1.0)).max() <= 1e-4


# --------------------------------------------------------------------------------------------------------------
def _rollout(g, wl, nom_dev):
    g.set_state(wl.broadcast_state.astype(np.float32), broadcast=True)
    s_start = g.step_counter
    g.step(nom_dev, wl.n_steps, cmd_hold=wl.cmd_hold)
    return s_start


@pytest.mark.parametrize("n_elite", [1, 7, 64, 211])
def test_r28_elite_selection_is_bit_exact_on_the_gpu_costs(cf, W, mp, n_elite):
    import torch
    wl = W.mppi(seed=5, n_ctrl=3, worlds_per_ctrl=211, horizon=4, cmd_hold=3, n_elite=n_elite)
    g = cf.Sim(wl.M, 1, wl.model, wl.params)
    g.reset(wl.seed)
    nom = torch.as_tensor(random_nominal(wl, 2), device="cuda")
    _rollout(g, wl, nom.clone())
    cost = g.cost().cpu().numpy()
    out = g.mppi_update(g.mppi_params(4, 3, n_elite, 0.5), nom.clone(), want_elites=True)
    assert np.array_equal(out["elites"].cpu().numpy(), mp.elite_select(cost, 3, n_elite))
    info = out["info"].cpu().numpy()
    thr = np.array([np.sort(cost[c * 211:(c + 1) * 211])[n_elite - 1] for c in range(3)])
    assert np.array_equal(info[3:12:4], thr) and np.array_equal(info[1:12:4], cost.reshape(3, -1).min(1))


def test_r28_selection_with_more_keys_than_the_register_resident_path_holds(cf, W, mp):
    """150 001 rollouts per controller: each thread's segment is longer than the 16 register-resident keys."""
    import torch
    wl = W.mppi(seed=12, n_ctrl=2, worlds_per_ctrl=150_001, horizon=3, cmd_hold=2, n_elite=1500)
    g = cf.Sim(wl.M, 1, wl.model, wl.params)
    g.reset(wl.seed)
    nom = torch.as_tensor(random_nominal(wl, 4), device="cuda")
    _rollout(g, wl, nom.clone())
    cost = g.cost().cpu().numpy()
    for n_elite in (1500, 4096):
        out = g.mppi_update(g.mppi_params(3, 2, n_elite, 0.5), nom.clone(), want_elites=True)
        assert np.array_equal(out["elites"].cpu().numpy(), mp.elite_select(cost, 2, n_elite))


def test_r28_ties_nan_and_infinities_follow_the_bit_pattern_rule(cf, W, mp):
    import torch
    wl = W.mppi(seed=6, n_ctrl=2, worlds_per_ctrl=1500, horizon=3, cmd_hold=2, n_elite=40)
    p = dict(wl.params, cost_w_pos=0.0, cost_w_vel=0.0, cost_w_term=0.0, cost_w_obs=0.0, cost_w_coll=0.0)
    g = cf.Sim(wl.M, 1, wl.model, p)
    g.reset(wl.seed)
    nom = torch.as_tensor(wl.cmds, device="cuda")
    _rollout(g, wl, nom.clone())
    rng = np.random.default_rng(0)
    crafted = rng.integers(0, 9, wl.M).astype(np.float32)          # heavy ties: ~330 rollouts per value and controller
    crafted[rng.integers(0, wl.M, 50)] = np.nan
    crafted[rng.integers(0, wl.M, 20)] = np.inf
    g.set_plan_state(cost_run=crafted)                             # all weights 0: J == the injected running cost
    got_cost = g.cost().cpu().numpy()
    assert np.array_equal(got_cost, crafted, equal_nan=True)      # (J = J_run + 0 |e|^2 turns a -0 into +0: not injected)
    for n_elite in (1, 40, 333, 1499, 1500):
        out = g.mppi_update(g.mppi_params(3, 2, n_elite, 1.0), nom.clone(), want_elites=True)
        assert np.array_equal(out["elites"].cpu().numpy(), mp.elite_select(got_cost, 2, n_elite)), n_elite


# --------------------------------------------------------------------------------------------------------------
def _check_update(out, ref, n_ctrl):
    info = out["info"].cpu().numpy()
    np.testing.assert_allclose(info[0:4 * n_ctrl:4], ref["score"], rtol=2e-5)
    np.testing.assert_allclose(info[1:4 * n_ctrl:4], ref["jmin"], rtol=0, atol=0)
    np.testing.assert_allclose(info[2:4 * n_ctrl:4], ref["wsum"], rtol=2e-5)
    gap = np.sort(ref["score"].astype(np.float32))
    if n_ctrl == 1 or gap[1] - gap[0] > 1e-4 * abs(gap[0]):        # the float32 argmin is unambiguous
        assert int(info.view(np.int32)[4 * n_ctrl]) == ref["best"]
        np.testing.assert_allclose(out["plan"].cpu().numpy(), ref["plan"], rtol=0, atol=5e-6)
    np.testing.assert_allclose(out["nominal"].cpu().numpy(), ref["nominal_next"], rtol=0, atol=5e-6)


@pytest.mark.parametrize("lam,shift,n_elite", [(0.5, 1, 9), (0.02, 0, 30), (50.0, 3, 1), (0.5, 6, 211)])
def test_r29_r32_update_matches_the_oracle_on_the_same_costs(cf, W, mp, lam, shift, n_elite):
    import torch
    wl = W.mppi(seed=7, n_ctrl=3, worlds_per_ctrl=211, horizon=6, cmd_hold=5, n_elite=n_elite)
    g = cf.Sim(wl.M, 1, wl.model, wl.params)
    g.reset(wl.seed)
    nom_np = random_nominal(wl, 3)
    nom = torch.as_tensor(nom_np, device="cuda")
    g.step(nom.clone(), 7, cmd_hold=7)                             # s_start != 0
    s_start = _rollout(g, wl, nom.clone())
    assert s_start == 7
    cost = g.cost().cpu().numpy()
    out = g.mppi_update(g.mppi_params(6, 5, n_elite, lam, shift), nom, want_elites=True)
    ref = oracle_update(mp, wl, cost, nom_np, s_start, n_elite=n_elite, lam=lam, shift=shift)
    assert np.array_equal(out["elites"].cpu().numpy(), ref["elites"])
    _check_update(out, ref, 3)


def test_closed_loop_iterations_track_the_oracle_chain(cf, cfo, W, mp):
    """cf_mppi_iterate x 5 with the nominal evolving on the device; every iteration is checked against the oracle
    rollout (costs) and the oracle update (on the GPU's float32 costs and the GPU's incoming nominal)."""
    import torch
    wl = W.mppi(seed=8, n_ctrl=2, worlds_per_ctrl=384, horizon=8, cmd_hold=5, n_elite=12)
    g, o = pair(cf, cfo, wl)
    x0 = torch.as_tensor(wl.broadcast_state.astype(np.float32), device="cuda")
    nom = torch.as_tensor(wl.cmds, device="cuda")
    mpar = g.mppi_params(8, 5, 12, wl.notes["lam"], 1)
    scores = []
    for it in range(5):
        nom_in = nom.cpu().numpy().copy()
        s_start = g.step_counter
        out = g.mppi_iterate(mpar, x0, nom, want_elites=True)
        cost = g.cost().cpu().numpy()
        o.set_state(wl.broadcast_state, broadcast=True)
        o.step(nom_in, wl.n_steps, cmd_hold=wl.cmd_hold)
        Jo = o.cost()
        assert (np.abs(cost - Jo) / np.maximum(np.abs(Jo), 1.0)).max() <= 1e-4, it
        ref = oracle_update(mp, wl, cost, nom_in, s_start, n_elite=12)
        assert np.array_equal(out["elites"].cpu().numpy(), ref["elites"]), it
        _check_update(out, ref, 2)
        scores.append(float(ref["score"].min()))
    assert g.step_counter == 5 * wl.n_steps and scores[-1] < scores[0]


def test_a_shard_of_controllers_reproduces_its_slice_of_the_full_run(cf, W):
    """Sharding by controllers (planner.py): rank 1 of 2 runs controllers 2, 3 with world_offset = 2 K_c and must get
    bit-identical costs, elite sets and warm-started nominals, and packing + selecting gives the full run's plan."""
    import torch
    from paper_2606_01478_b200 import planner
    full = W.mppi(seed=21, n_ctrl=4, worlds_per_ctrl=320, horizon=5, cmd_hold=3, n_elite=10)
    nom_np = random_nominal(full, 6)
    x0 = torch.as_tensor(full.broadcast_state.astype(np.float32), device="cuda")
    gf = cf.Sim(full.M, 1, full.model, full.params)
    gf.reset(full.seed)
    nom_f = torch.as_tensor(nom_np, device="cuda")
    of = gf.mppi_iterate(gf.mppi_params(5, 3, 10, 0.5, 1), x0, nom_f, want_elites=True)
    cost_f, el_f, plan_f = gf.cost().cpu().numpy(), of["elites"].cpu().numpy().copy(), of["plan"].cpu().numpy().copy()
    best_f = int(of["info"].cpu().numpy().view(np.int32)[16])
    rows = []
    for rank in range(2):
        gs = cf.Sim(640, 1, full.model, dict(full.params, n_ctrl=2, world_offset=rank * 640))
        gs.reset(full.seed)
        nom_s = torch.as_tensor(nom_np[2 * rank:2 * rank + 2].copy(), device="cuda")
        os_ = gs.mppi_iterate(gs.mppi_params(5, 3, 10, 0.5, 1), x0, nom_s, want_elites=True)
        sl = slice(rank * 640, (rank + 1) * 640)
        assert np.array_equal(gs.cost().cpu().numpy(), cost_f[sl])
        assert np.array_equal(os_["elites"].cpu().numpy(), el_f[2 * rank:2 * rank + 2])
        assert np.array_equal(nom_s.cpu().numpy(), nom_f.cpu().numpy()[2 * rank:2 * rank + 2])
        mp_ = gs.mppi_params(5, 3, 10, 0.5, 1)
        rows.append(gs.mppi_pack_best(mp_, os_["info"], os_["plan"], rank * 2).clone())
        plan1, score1, gidx1 = planner.select_global_plan(gs, mp_, os_, rank)          # world size 1: the shard's own best
        assert torch.equal(plan1, os_["plan"]) and int(gidx1) == int(rows[-1][1])
    from oracle import mppi as omppi
    for order in ([0, 1], [1, 0]):                                                     # the winner does not depend on the row order
        stacked = torch.stack([rows[k] for k in order]).contiguous()
        best = gs.mppi_select(stacked, 5).cpu().numpy()
        assert np.array_equal(best, stacked.cpu().numpy()[omppi.select_rows(stacked.cpu().numpy())])
        assert int(best[1]) == best_f and np.array_equal(best[2:].reshape(-1, 4), plan_f)
    # ties -> lowest global controller index, NaN last, -0 before +0 (R31 / R28 key order), against the oracle's rule
    W_ = 2 + 4 * 5
    rng = np.random.default_rng(0)
    for trial in range(20):
        n = int(rng.integers(1, 9))
        r = rng.normal(size=(n, W_)).astype(np.float32)
        r[:, 0] = rng.choice(np.array([1.0, 1.0, -0.0, 0.0, np.nan, 2.5], dtype=np.float32), n)
        r[:, 1] = rng.permutation(16)[:n]
        got = gs.mppi_select(torch.as_tensor(r, device="cuda"), 5).cpu().numpy()
        assert np.array_equal(got, r[omppi.select_rows(r)], equal_nan=True), (trial, r[:, :2])


def test_planner_argument_and_state_errors(cf, W):
    import torch
    wl = W.mppi(seed=9, n_ctrl=2, worlds_per_ctrl=64, horizon=4, cmd_hold=2, n_elite=4)
    g = cf.Sim(wl.M, 1, wl.model, wl.params)
    g.reset(wl.seed)
    nom = torch.as_tensor(wl.cmds, device="cuda")
    with pytest.raises(cf.CfError) as e:                           # no rollout yet
        g.mppi_update(g.mppi_params(4, 2, 4, 0.5), nom)
    assert e.value.code == cf.E_STATE
    _rollout(g, wl, nom)
    g.mppi_update(g.mppi_params(4, 2, 4, 0.5), nom.clone())
    with pytest.raises(cf.CfError) as e:                           # horizon does not match the rollout
        g.mppi_update(g.mppi_params(2, 4, 4, 0.5), nom[:, :2].contiguous())
    assert e.value.code == cf.E_STATE
    g.step(nom, 2, cmd_hold=2)                                     # a second cf_step: the rollout is no longer fresh
    with pytest.raises(cf.CfError) as e:
        g.mppi_update(g.mppi_params(4, 2, 4, 0.5), nom.clone())
    assert e.value.code == cf.E_STATE
    for bad in (dict(n_elite=0), dict(n_elite=65), dict(lam=0.0), dict(shift=5)):
        kw = dict(horizon=4, cmd_hold=2, n_elite=4, lam=0.5, shift=1)
        kw.update(bad)
        with pytest.raises(cf.CfError) as e:
            g.mppi_update(g.mppi_params(**kw), nom.clone())
        assert e.value.code == cf.E_ARG, bad
    with pytest.raises(cf.CfError) as e:                           # the rollout cost needs single-drone worlds
        cf.Sim(4, 2, wl.model, dict(wl.params, n_ctrl=1, worlds_per_ctrl=0))
    assert e.value.code == cf.E_UNSUPPORTED
    with pytest.raises(cf.CfError) as e:                           # more worlds than nominal sequences
        cf.Sim(wl.M + 1, 1, wl.model, wl.params)
    assert e.value.code == cf.E_SHAPE


def test_full_size_planner_iteration_sampled_against_the_oracle(cf, cfo, W, mp):
    """The bench configuration (5 x 100 000 rollouts, 25 knots x 10 steps, 1000 elites per controller): exact elite
    sets on the GPU costs, oracle update, and sampled rollouts re-simulated one by one by the oracle."""
    import torch
    wl = W.mppi()
    g = cf.Sim(wl.M, 1, wl.model, wl.params)
    g.reset(wl.seed)
    x0 = torch.as_tensor(wl.broadcast_state.astype(np.float32), device="cuda")
    nom_np = random_nominal(wl, 5, amp=0.1)
    nom = torch.as_tensor(nom_np, device="cuda")
    n = wl.notes
    mpar = g.mppi_params(n["horizon"], wl.cmd_hold, n["n_elite"], n["lam"], n["shift"])
    out = g.mppi_iterate(mpar, x0, nom, want_elites=True)
    cost = g.cost().cpu().numpy()
    state = g.get_state().cpu().numpy()
    assert np.isfinite(cost).all()
    ref = oracle_update(mp, wl, cost, nom_np, 0)
    assert np.array_equal(out["elites"].cpu().numpy(), ref["elites"])
    _check_update(out, ref, n["n_ctrl"])
    rng = np.random.default_rng(1)
    sample = np.concatenate([[0, 31, 32, wl.M - 1, 99_999, 100_000], rng.integers(0, wl.M, 42),
                             ref["elites"][3][:8] + 300_000])
    for w in sample:
        o = cfo.OracleSim(1, 1, wl.model, dict(wl.params, world_offset=int(w), n_ctrl=1))   # a one-world shard ...
        o.reset(wl.seed)
        o.set_state(wl.broadcast_state, broadcast=True)
        c = int(w) // wl.params["worlds_per_ctrl"]                                           # ... of controller c
        o.step(nom_np[c:c + 1].copy(), wl.n_steps, cmd_hold=wl.cmd_hold)
        assert rel_state_err(state[:, w:w + 1], o.get_state()) <= 1e-4, w
        Jo = o.cost()[0]
        assert abs(cost[w] - Jo) <= 1e-4 * max(abs(Jo), 1.0), w
