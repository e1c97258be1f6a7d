"""float64 ORACLE of the sampling-based planner around the planning rollout (hybrid iCEM / MPPI update).

TEST INFRASTRUCTURE ONLY (see oracle/cfo.h): imported by tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs; shares nothing with paper_2606_01478_b200/.

What the paper fixes ("Model Predictive Path Integral"): a hybrid of iCEM and MPPI; several
independent controllers run in parallel and the best control sequence is selected at each step; each controller
truncates to the top 1 % of trajectories (elites), uses temporally correlated noise, and warm-starts its sampling
from the previous mean; the mean across the best samples is an exponential weighting over all elites, as in MPPI;
500 k parallel rollouts, 25-step horizon, 50 Hz.  The parameters are in a codebase that is not available, and no
equation is printed, so everything below is a reading (R25-R33).  The steps, in order:

  R25  noise: eps_0 = z_0, eps_t = beta eps_{t-1} + sqrt(1 - beta^2) z_t, z_t ~ N(0, I_4) from the Philox NOISE stream
       (counter (world, 0, step at which the command is formed, 3)); implemented in oracle/cfo.c (the rollout).
  R26  command of rollout k of controller c at knot t:  u_k[t] = clip(nominal_c[t] + sigma * eps_k[t], lo, hi).
  R27  cost J_k (oracle/cfo.c, CFO_AUX_COST).
  R28  elites E_c: the n_elite rollouts of controller c with the smallest (cost, world index), the cost compared as a
       float32 in IEEE total order with NaN last (an exact integer rule on the float32 bit pattern).
  R29  weights w_k = exp(-(J_k - J_min,c) / lambda), J_min,c = min over E_c.
  R30  mean_c[t] = sum_{k in E_c} w_k u_k[t] / sum_k w_k   (u_k[t]: the clipped command the rollout applied).
  R31  score S_c = sum w_k J_k / sum w_k;  best controller c* = argmin_c S_c compared in float32, ties -> lowest c.
  R32  plan = mean_{c*};  warm start: nominal'_c[t] = mean_c[min(t + shift, H - 1)].

Parity pins: tests/test_oracle_mppi.py (hand-worked tiny cases, limits lambda -> 0 / infinity, shift, tie-breaks,
bit-pattern ordering, regenerated commands == commands the rollout applied, AR(1) moments, cost closed forms).
"""
from __future__ import annotations

import numpy as np

from . import cfo

STREAM_NOISE = 3


def cost_key(cost_f32) -> np.ndarray:
    """R28: uint32 key whose unsigned order is the IEEE total order of the float32 costs, NaN (any sign) last."""
    c = np.ascontiguousarray(cost_f32, dtype=np.float32)
    bits = c.view(np.uint32)
    neg = (bits >> np.uint32(31)).astype(bool)
    key = np.where(neg, ~bits, bits | np.uint32(0x80000000)).astype(np.uint32)
    key[np.isnan(c)] = np.uint32(0xFFFFFFFF)
    return key


def elite_select(cost_f32, n_ctrl: int, n_elite: int) -> np.ndarray:
    """R28.  cost_f32: [n_ctrl * K_c].  Returns int64 [n_ctrl][n_elite]: indices local to the controller, ascending."""
    key = cost_key(cost_f32).reshape(n_ctrl, -1)
    K_c = key.shape[1]
    assert 1 <= n_elite <= K_c
    out = np.empty((n_ctrl, n_elite), dtype=np.int64)
    for c in range(n_ctrl):
        order = np.lexsort((np.arange(K_c), key[c]))     # primary: key, secondary: index
        out[c] = np.sort(order[:n_elite])
    return out


def noise_chain(seed: int, world_global: int, s_start: int, cmd_hold: int, horizon: int, beta: float) -> np.ndarray:
    """R25 restated outside the rollout: eps[t][4] of one rollout whose first command is formed at step s_start."""
    eps = np.empty((horizon, 4))
    gain = np.sqrt(1.0 - beta * beta)
    for t in range(horizon):
        r = cfo.philox(seed, (world_global & 0xFFFFFFFF, 0, (s_start + t * cmd_hold) & 0xFFFFFFFF, STREAM_NOISE))
        z = np.array(cfo.normal_pair(r[0], r[1]) + cfo.normal_pair(r[2], r[3]))
        eps[t] = z if t == 0 else beta * eps[t - 1] + gain * z
    return eps


def applied_commands(seed, world_global, s_start, cmd_hold, nominal_c, sigma, beta, lo, hi) -> np.ndarray:
    """R26: the clipped commands u[t][4] rollout `world_global` applied.  nominal_c: float32 [H][4]."""
    nominal_c = np.asarray(nominal_c, dtype=np.float32).astype(np.float64)
    eps = noise_chain(seed, world_global, s_start, cmd_hold, nominal_c.shape[0], beta)
    return np.clip(nominal_c + np.asarray(sigma, dtype=np.float64) * eps, np.asarray(lo, dtype=np.float64),
                   np.asarray(hi, dtype=np.float64))


def update(cost_f32, nominal, *, seed: int, world_offset: int, worlds_per_ctrl: int, s_start: int, cmd_hold: int,
           sigma, beta: float, lo, hi, n_elite: int, lam: float, shift: int = 1) -> dict:
    """R28-R32 for all controllers.  cost_f32: [n_ctrl * worlds_per_ctrl] float32 costs of the rollouts (world order);
    nominal: float32 [n_ctrl][H][4], the sequences the rollouts were sampled around."""
    nominal = np.asarray(nominal, dtype=np.float32)
    n_ctrl, H, _ = nominal.shape
    cost_f32 = np.ascontiguousarray(cost_f32, dtype=np.float32)
    assert cost_f32.size == n_ctrl * worlds_per_ctrl
    elites = elite_select(cost_f32, n_ctrl, n_elite)
    mean = np.zeros((n_ctrl, H, 4))
    score = np.zeros(n_ctrl)
    jmin = np.zeros(n_ctrl)
    wsum = np.zeros(n_ctrl)
    for c in range(n_ctrl):
        J = cost_f32[c * worlds_per_ctrl + elites[c]].astype(np.float64)
        jmin[c] = J.min()
        w = np.exp(-(J - jmin[c]) / lam)                                  # R29
        wsum[c] = w.sum()
        for k, wk in zip(elites[c], w):
            wg = world_offset + c * worlds_per_ctrl + int(k)
            mean[c] += wk * applied_commands(seed, wg, s_start, cmd_hold, nominal[c], sigma, beta, lo, hi)
        mean[c] /= wsum[c]                                                # R30
        score[c] = (w * J).sum() / wsum[c]                                # R31
    best = int(np.argmin(score.astype(np.float32)))                       # first minimum = lowest c on ties
    idx = np.minimum(np.arange(H) + shift, H - 1)
    return dict(elites=elites, mean=mean, score=score, jmin=jmin, wsum=wsum, best=best, plan=mean[best].copy(),
                nominal_next=mean[:, idx, :].copy())


def select_rows(rows) -> int:
    """R31 across shards: rows [n][2 + 4 H] of (score, global controller index, plan...) -> index of the winning row:
    smallest score compared as a float32 in IEEE total order with NaN last (the R28 key), ties -> smallest controller index."""
    rows = np.asarray(rows, dtype=np.float32).reshape(len(rows), -1)
    key = cost_key(rows[:, 0])
    return int(np.lexsort((rows[:, 1], key))[0])
