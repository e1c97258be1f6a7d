"""Pins of the planner oracle (oracle/mppi.py + the planning-rollout parts of oracle/cfo.c): DESIGN.md R25-R32,
PAPER.md:L465-L471.  Nothing here re-types the oracle's formulas: the checks are moments of the AR(1) process,
polynomial-sum closed forms on a drifting hover, brute force over recorded positions, hand-worked tiny selections,
the limits lambda -> 0 / infinity, invariances, and agreement of two separately written code paths
(commands applied inside the C rollout vs. regenerated in Python from the counter-based generator).
"""
import math

import numpy as np
import pytest

M_, G_ = 0.027, 9.81
HOVER = float(np.float32(M_ * G_))


@pytest.fixture(scope="module")
def mp():
    from oracle import mppi
    return mppi


def ab_start(v=(1.0, 0.0, 0.0), p=(0.0, 0.0, 1.0)):
    x = np.zeros(13)
    x[:3] = p
    x[6:9] = v
    x[12] = HOVER
    return x


def plan_sim(cfo, M, **ov):
    base = dict(integrator=cfo.EULER, iface=cfo.IF_ATTITUDE, f_phys=500.0, f_att=500.0, init_mode=0,
                cmd_source=cfo.CMD_NOMINAL_PLUS_NOISE, noise_sigma=[0.15, 0.15, 0.05, 0.03])
    base.update(ov)
    sim = cfo.OracleSim(M, 1, cfo.MODEL_AB, base)
    return sim


def hover_nominal(n_ctrl, H):
    nom = np.zeros((n_ctrl, H, 4), dtype=np.float32)
    nom[..., 3] = HOVER
    return nom


# ------------------------------------------------------------------------------------------------------------
# R25: temporally correlated noise
def test_r25_first_draw_after_rearm_is_the_plain_normal_and_beta0_is_white(cfo):
    seed, M = 11, 7
    for beta in (0.0, 0.6):
        sim = plan_sim(cfo, M, noise_beta=beta, world_offset=5)
        sim.reset(seed)
        assert np.isnan(sim.eps()).all()                       # nothing drawn since the re-arm
        sim.step(hover_nominal(1, 3), 3, cmd_hold=1)
        sim.set_state(ab_start(), broadcast=True)              # re-arm: the chain starts afresh
        assert np.isnan(sim.eps()).all()
        s0 = int(sim.counters()[0])
        z = []
        for t in range(3):
            sim.step(hover_nominal(1, 1), 1, cmd_hold=1)
            zt = np.empty((4, M))
            for w in range(M):
                r = cfo.philox(seed, (w + 5, 0, s0 + t, 3))
                zt[:, w] = cfo.normal_pair(r[0], r[1]) + cfo.normal_pair(r[2], r[3])
            z.append(zt)
            if t == 0 or beta == 0.0:
                np.testing.assert_allclose(sim.eps(), zt, rtol=0, atol=1e-15)
        if beta > 0:      # after three draws: beta^2 z0 + beta g z1 + g z2 (unrolled recursion), g^2 = 1 - beta^2
            g = math.sqrt(1 - beta * beta)
            np.testing.assert_allclose(sim.eps(), beta * beta * z[0] + beta * g * z[1] + g * z[2], atol=1e-14)


def test_r25_ar1_is_stationary_with_unit_variance_and_lag_correlation_beta(cfo):
    M, H, beta = 40000, 12, 0.8
    sim = plan_sim(cfo, M, noise_beta=beta)
    sim.reset(3)
    e = []
    for t in range(H):
        sim.step(hover_nominal(1, 1), 1, cmd_hold=1)
        e.append(sim.eps().copy())
    e = np.array(e)                                            # [H][4][M]
    n = 4 * M
    for t in (0, 1, 5, H - 1):                                 # unit variance at EVERY knot, the first included
        v = e[t].var()
        assert abs(v - 1.0) < 4 * math.sqrt(2.0 / n), (t, v)
        assert abs(e[t].mean()) < 4 / math.sqrt(n)
    for lag in (1, 2, 3):
        c = (e[4] * e[4 + lag]).mean()
        assert abs(c - beta ** lag) < 4 * math.sqrt((1 + beta ** (2 * lag)) / n), (lag, c)


# ------------------------------------------------------------------------------------------------------------
# R26: per-controller nominal + clip; the commands the rollout applies can be regenerated from the counters alone
def test_r26_regenerated_commands_equal_the_commands_the_rollout_applied(cfo, mp):
    seed, n_ctrl, Kc, H, hold, beta = 5, 3, 4, 5, 3, 0.5
    sigma, lo, hi = [0.4, 0.15, 0.05, 0.05], [-0.5, -0.5, -math.pi, 0.05], [0.5, 0.5, math.pi, 0.55]
    rng = np.random.default_rng(0)
    nom = hover_nominal(n_ctrl, H)
    nom[..., 0] = rng.uniform(-0.4, 0.4, (n_ctrl, H))          # different per controller and knot; roll will clip
    nom[..., 3] += rng.uniform(-0.05, 0.05, (n_ctrl, H)).astype(np.float32)
    sim = plan_sim(cfo, n_ctrl * Kc, noise_beta=beta, noise_sigma=sigma, cmd_lo=lo, cmd_hi=hi, n_ctrl=n_ctrl,
                   worlds_per_ctrl=Kc, world_offset=0)
    sim.reset(seed)
    sim.step(hover_nominal(n_ctrl, 1), 7, cmd_hold=7)          # move the step counter off zero
    sim.set_state(ab_start(), broadcast=True)
    s_start = int(sim.counters()[0])
    applied = np.empty((H, 4, n_ctrl * Kc))
    for t in range(H):                                         # knot by knot: split == fused, so this is the rollout
        sim.step(nom[:, t:t + 1], hold, cmd_hold=hold)
        applied[t] = sim.ctrl()[6:10]                          # held attitude command planes
    clipped = 0
    for w in range(n_ctrl * Kc):
        u = mp.applied_commands(seed, w, s_start, hold, nom[w // Kc], sigma, beta, lo, hi)
        np.testing.assert_allclose(applied[:, :, w], u, rtol=0, atol=1e-14)
        clipped += int((np.abs(u[:, 0]) == 0.5).sum())
    assert clipped > 0                                         # the clip was exercised
    # and the fused rollout gives the same final state as the knot-by-knot one
    sim2 = plan_sim(cfo, n_ctrl * Kc, noise_beta=beta, noise_sigma=sigma, cmd_lo=lo, cmd_hi=hi, n_ctrl=n_ctrl,
                    worlds_per_ctrl=Kc)
    sim2.reset(seed)
    sim2.step(hover_nominal(n_ctrl, 1), 7, cmd_hold=7)
    sim2.set_state(ab_start(), broadcast=True)
    sim2.step(nom, H * hold, cmd_hold=hold)
    assert np.array_equal(sim2.get_state(), sim.get_state())
    assert np.array_equal(sim2.eps(), sim.eps())


def test_r26_controller_index_is_local_to_the_shard_noise_is_global_and_the_range_is_checked(cfo):
    sim = plan_sim(cfo, 8, n_ctrl=2, worlds_per_ctrl=4, world_offset=40, noise_sigma=[0, 0, 0, 0])
    sim.reset(1)
    nom = hover_nominal(2, 1)
    nom[1, 0, 0] = 0.25                                        # local worlds 4..7 = this shard's controller 1
    sim.step(nom, 1, cmd_hold=1)
    np.testing.assert_allclose(sim.ctrl()[6], [0, 0, 0, 0, 0.25, 0.25, 0.25, 0.25])
    # a shard reproduces the slice of the full run: the noise is keyed by the global world index
    full = plan_sim(cfo, 16, n_ctrl=4, worlds_per_ctrl=4); full.reset(2)
    part = plan_sim(cfo, 8, n_ctrl=2, worlds_per_ctrl=4, world_offset=8); part.reset(2)
    nom4 = hover_nominal(4, 3); nom4[:, :, 1] = 0.1 * np.arange(4)[:, None]
    full.step(nom4, 3, cmd_hold=1); part.step(nom4[2:].copy(), 3, cmd_hold=1)
    assert np.array_equal(full.get_state()[:, 8:], part.get_state()) and np.array_equal(full.eps()[:, 8:], part.eps())
    bad = plan_sim(cfo, 9, n_ctrl=2, worlds_per_ctrl=4)
    bad.reset(1)
    rc, _ = bad.step(nom, 1, cmd_hold=1, check=False)
    assert rc == -2


# ------------------------------------------------------------------------------------------------------------
# R27: rollout cost
def test_r27_running_and_terminal_cost_closed_form_on_a_drifting_hover(cfo):
    n, h, vx = 60, 1 / 500.0, 1.5
    goal, wp, wv, wt = np.array([2.0, 0.3, 1.4]), 1.7, 0.05, 9.0
    sim = plan_sim(cfo, 2, noise_sigma=[0, 0, 0, 0], cost_on=1, cost_goal=goal, cost_w_pos=wp, cost_w_vel=wv,
                   cost_w_term=wt)
    sim.reset(1)
    sim.set_state(ab_start(v=(vx, 0, 0)), broadcast=True)
    sim.step(hover_nominal(1, 1), n, cmd_hold=n)
    # level hover drifts at constant velocity: p_k = p0 + k h v, so the sums over k are polynomial sums
    a, b = 0.0 - goal[0], h * vx
    s_x = n * a * a + a * b * n * (n + 1) + b * b * n * (n + 1) * (2 * n + 1) / 6
    run = h * (wp * (s_x + n * ((0 - goal[1]) ** 2 + (1 - goal[2]) ** 2)) + wv * n * vx * vx)
    pT = np.array([n * h * vx, 0.0, 1.0])
    fused = sim.cost_run().copy()
    np.testing.assert_allclose(fused, run, rtol=1e-6)
    np.testing.assert_allclose(sim.cost(), run + wt * ((pT - goal) ** 2).sum(), rtol=1e-6)
    # a re-arm zeroes the running part; a split run accumulates the same total
    sim.set_state(ab_start(v=(vx, 0, 0)), broadcast=True)
    assert (sim.cost_run() == 0).all()
    for m in (7, 20, 33):
        sim.step(hover_nominal(1, 1), m, cmd_hold=m)
    assert np.array_equal(sim.cost_run(), fused)


@pytest.mark.parametrize("y_off,expect", [(0.60, "free"), (0.40, "near"), (0.10, "hit")])
def test_r27_obstacle_clearance_and_collision_terms(cfo, y_off, expect):
    n, h, vx, r, d_safe, wo, wc = 250, 1 / 500.0, 2.0, 0.25, 0.2, 300.0, 1000.0
    obst = np.zeros((8, 4))
    obst[0] = [0.5, y_off, 1.0, r]
    obst[1] = [9.0, 9.0, 9.0, 0.1]
    sim = plan_sim(cfo, 1, noise_sigma=[0, 0, 0, 0], cost_on=1, n_obstacles=2, obstacles=obst, cost_w_obs=wo,
                   cost_d_safe=d_safe, cost_w_coll=wc)
    sim.reset(1)
    sim.set_state(ab_start(v=(vx, 0, 0)), broadcast=True)
    rec = sim.step(hover_nominal(1, 1), n, cmd_hold=n, record_every=1)
    p = rec[:, :3, 0]                                              # brute force over the recorded positions
    d_min = min(np.sqrt(((p - obst[j, :3]) ** 2).sum(1)).min() - obst[j, 3] for j in range(2))
    J = sim.cost()[0]
    if expect == "free":
        assert d_min > d_safe and J == 0.0
    elif expect == "near":
        assert 0 < d_min < d_safe
        assert J == pytest.approx(wo * (d_safe - d_min) ** 2, rel=1e-9)
    else:
        assert d_min < 0
        assert J == pytest.approx(wo * (d_safe - d_min) ** 2 + wc, rel=1e-9)
    assert sim.min_dist()[0] == pytest.approx(d_min, abs=1e-12)


# ------------------------------------------------------------------------------------------------------------
# R28: elite selection is an exact rule on the float32 bit patterns
def test_r28_total_order_of_special_values_and_nan_last(mp):
    vals = np.array([np.nan, np.inf, 1.0, 1e-45, 0.0, -0.0, -1.0, -np.inf], dtype=np.float32)
    key = mp.cost_key(vals)
    assert list(np.argsort(key, kind="stable")) == [7, 6, 5, 4, 3, 2, 1, 0]
    neg_nan = np.array([0xFFC00000], dtype=np.uint32).view(np.float32)
    assert mp.cost_key(neg_nan)[0] == 0xFFFFFFFF                   # NaN of either sign sorts last
    x = np.random.default_rng(0).standard_normal(5000).astype(np.float32)
    k = mp.cost_key(x)
    o = np.argsort(x, kind="stable")
    assert (np.diff(k[o].astype(np.int64)) >= 0).all()             # monotone in the value


def test_r28_hand_worked_selection_with_ties_goes_to_the_lowest_index(mp):
    cost = np.array([3, 1, 2, 1, 5, 1,    # controller 0: three ones (indices 1, 3, 5), n_elite = 2 -> {1, 3}
                     0, 0, 0, 0, 0, 0],   # controller 1: all equal -> {0, 1}
                    dtype=np.float32)
    assert mp.elite_select(cost, 2, 2).tolist() == [[1, 3], [0, 1]]
    assert mp.elite_select(cost, 2, 4).tolist() == [[1, 2, 3, 5], [0, 1, 2, 3]]
    assert mp.elite_select(cost, 2, 6).tolist() == [[0, 1, 2, 3, 4, 5]] * 2


def test_r28_selection_matches_brute_force_on_heavily_tied_costs(mp):
    rng = np.random.default_rng(1)
    for trial in range(20):
        n_ctrl, Kc = 3, 57
        cost = rng.integers(0, 6, n_ctrl * Kc).astype(np.float32)
        cost[rng.integers(0, n_ctrl * Kc, 4)] = np.nan
        n_elite = int(rng.integers(1, Kc + 1))
        got = mp.elite_select(cost, n_ctrl, n_elite)
        for c in range(n_ctrl):
            cc = cost[c * Kc:(c + 1) * Kc]
            pairs = sorted(range(Kc), key=lambda i: (math.inf if math.isnan(cc[i]) else float(cc[i]),
                                                     math.isnan(cc[i]), i))
            assert got[c].tolist() == sorted(pairs[:n_elite])


# ------------------------------------------------------------------------------------------------------------
# R29-R32: weights, mean, score, best controller, warm start
_UPD = dict(seed=9, world_offset=0, worlds_per_ctrl=4, s_start=17, cmd_hold=2, sigma=[0.15, 0.15, 0.05, 0.03],
            beta=0.5, lo=[-0.5, -0.5, -math.pi, 0.05], hi=[0.5, 0.5, math.pi, 0.55])


def _u(mp, c, k, nominal):
    a = _UPD
    return mp.applied_commands(a["seed"], c * 4 + k, a["s_start"], a["cmd_hold"], nominal[c], a["sigma"], a["beta"],
                               a["lo"], a["hi"])


def test_r29_r32_hand_worked_two_elites(mp):
    H = 3
    nominal = hover_nominal(1, H)
    cost = np.array([3, 1, 2, 5], dtype=np.float32)               # elites {1, 2}; lambda = 1: w = (1, e^-1)
    out = mp.update(cost, nominal, n_elite=2, lam=1.0, shift=1, **_UPD)
    assert out["elites"].tolist() == [[1, 2]]
    w2 = math.exp(-1.0)
    mean = (_u(mp, 0, 1, nominal) + w2 * _u(mp, 0, 2, nominal)) / (1 + w2)
    np.testing.assert_allclose(out["mean"][0], mean, rtol=1e-14)
    assert out["score"][0] == pytest.approx((1 + 2 * w2) / (1 + w2), rel=1e-14)
    assert out["jmin"][0] == 1.0 and out["best"] == 0
    np.testing.assert_allclose(out["plan"], mean, rtol=1e-14)
    np.testing.assert_allclose(out["nominal_next"][0], mean[[1, 2, 2]], rtol=1e-14)   # shifted, last knot repeated
    out0 = mp.update(cost, nominal, n_elite=2, lam=1.0, shift=0, **_UPD)
    np.testing.assert_allclose(out0["nominal_next"][0], mean, rtol=1e-14)


def test_r29_r31_limits_invariances_and_best_controller(mp):
    H, n_ctrl = 4, 2
    rng = np.random.default_rng(3)
    nominal = hover_nominal(n_ctrl, H)
    nominal[..., :2] = rng.uniform(-0.2, 0.2, (n_ctrl, H, 2)).astype(np.float32)
    cost = np.array([4, 8, 6, 16,  7, 3, 5, 9], dtype=np.float32)
    big = mp.update(cost, nominal, n_elite=3, lam=1e15, **_UPD)   # lambda -> infinity: plain average of the elites
    for c, el in enumerate([[0, 1, 2], [0, 1, 2]]):
        np.testing.assert_allclose(big["mean"][c], np.mean([_u(mp, c, k, nominal) for k in el], axis=0), rtol=1e-12)
    np.testing.assert_allclose(big["score"], [6.0, 5.0], rtol=1e-12)
    assert big["best"] == 1
    tiny = mp.update(cost, nominal, n_elite=3, lam=1e-9, **_UPD)  # lambda -> 0: the best sample alone
    np.testing.assert_allclose(tiny["mean"][0], _u(mp, 0, 0, nominal), rtol=1e-12)
    np.testing.assert_allclose(tiny["mean"][1], _u(mp, 1, 1, nominal), rtol=1e-12)
    np.testing.assert_allclose(tiny["score"], [4.0, 3.0], rtol=1e-12)
    a = mp.update(cost, nominal, n_elite=3, lam=2.0, **_UPD)      # a common cost offset changes nothing but the score
    b = mp.update(cost + np.float32(64), nominal, n_elite=3, lam=2.0, **_UPD)
    np.testing.assert_allclose(a["mean"], b["mean"], rtol=1e-13)
    np.testing.assert_allclose(b["score"] - a["score"], 64.0, rtol=1e-12)
    same = mp.update(np.ones(8, dtype=np.float32), nominal, n_elite=2, lam=1.0, **_UPD)
    assert same["best"] == 0                                       # score tie -> lowest controller
    zero = dict(_UPD, sigma=[0, 0, 0, 0])                          # no noise: every sample is the nominal
    z = mp.update(cost, nominal, n_elite=3, lam=0.7, **zero)
    np.testing.assert_allclose(z["mean"], nominal.astype(np.float64), rtol=1e-15)


# ------------------------------------------------------------------------------------------------------------
def test_closed_loop_planner_lowers_the_cost_and_avoids_the_obstacle(cfo, mp):
    """Soft pin: iterating rollout -> update on the oracle steers around a sphere blocking the straight line."""
    n_ctrl, Kc, H, hold, n_elite, lam, beta = 2, 96, 12, 10, 8, 0.05, 0.7
    sigma, lo, hi = [0.25, 0.25, 0.0, 0.03], [-0.5, -0.5, -math.pi, 0.05], [0.5, 0.5, math.pi, 0.55]
    obst = np.zeros((8, 4))
    obst[0] = [0.35, 0.0, 1.0, 0.12]
    ov = dict(noise_beta=beta, noise_sigma=sigma, cmd_lo=lo, cmd_hi=hi, n_ctrl=n_ctrl, worlds_per_ctrl=Kc,
              n_obstacles=1, obstacles=obst, cost_on=1, cost_goal=[0.8, 0.0, 1.0], cost_w_pos=1.0, cost_w_vel=0.02,
              cost_w_term=20.0, cost_w_obs=400.0, cost_d_safe=0.1, cost_w_coll=100.0)
    sim = plan_sim(cfo, n_ctrl * Kc, **ov)
    sim.reset(2)
    x0 = ab_start(v=(1.5, 0, 0))
    nominal = hover_nominal(n_ctrl, H)
    scores = []
    for it in range(8):
        sim.set_state(x0, broadcast=True)
        s_start = int(sim.counters()[0])
        sim.step(nominal, H * hold, cmd_hold=hold)
        cost = sim.cost().astype(np.float32)
        out = mp.update(cost, nominal, seed=2, world_offset=0, worlds_per_ctrl=Kc, s_start=s_start, cmd_hold=hold,
                        sigma=sigma, beta=beta, lo=lo, hi=hi, n_elite=n_elite, lam=lam, shift=0)
        scores.append(out["score"].min())
        nominal = out["nominal_next"].astype(np.float32)
    # the noise-free rollout of the final plan vs. of the hover nominal
    def plan_cost(seq):
        s = plan_sim(cfo, 1, **dict(ov, noise_sigma=[0, 0, 0, 0], n_ctrl=1, worlds_per_ctrl=0))
        s.reset(2)
        s.set_state(x0, broadcast=True)
        s.step(seq[None], H * hold, cmd_hold=hold)
        return s.cost()[0], s.min_dist()[0]
    J_plan, d_plan = plan_cost(out["plan"].astype(np.float32))
    J_hover, d_hover = plan_cost(hover_nominal(1, H)[0])
    assert d_hover < 0 < d_plan                                    # hover flies through the sphere, the plan does not
    assert J_plan < 0.5 * J_hover
    assert scores[-1] < scores[0]
