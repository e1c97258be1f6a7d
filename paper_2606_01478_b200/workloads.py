"""Seeded synthetic workloads shaped like the paper's.

This module serves BOTH the CUDA path and the float64 oracle and therefore holds none of the
method's arithmetic: it only lists configuration values (BASELINE.json:configs)
and draws harness-side random inputs (commands, targets, obstacle scenes) with numpy's own
generator.  Random numbers the *method* draws (reset, parameter jitter, disturbances, command
noise) are drawn independently by each side from its own Philox4x32-10 implementation.

The paper measures on its own synthetic scaling sweeps (single drone x 2^k
worlds, swarms of 4000, 500k-rollout planning batches); these inputs stand in for them.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

MODEL_FP, MODEL_AB = 0, 1
EULER, RK4 = 0, 1
IF_ROTOR, IF_TORQUE, IF_ATTITUDE, IF_POSITION = 0, 1, 2, 3
CMD_BUFFER, CMD_NOMINAL_PLUS_NOISE = 0, 1

REPORT_SEED = 20260601
MASS, G = 0.027, 9.81


@dataclass
class Workload:
    name: str
    M: int
    N: int
    model: int
    params: dict                      # overrides of the library defaults, same keys in both bindings
    seed: int
    n_steps: int
    cmd_hold: int
    record_every: int
    cmds: np.ndarray | None           # float32 [K][M*N][4] or [K][4] (nominal + noise); None = make on device
    broadcast_state: np.ndarray | None = None   # [D] -> cf_set_state(broadcast=1) after reset
    notes: dict = field(default_factory=dict)

    @property
    def MN(self) -> int:
        return self.M * self.N

    @property
    def D(self) -> int:
        return 17 if self.model == MODEL_FP else 13

    @property
    def n_cmds(self) -> int:
        return -(-self.n_steps // self.cmd_hold)

    @property
    def drone_steps(self) -> int:
        return self.MN * self.n_steps

    def n_records(self, s0: int = 0) -> int:
        if self.record_every <= 0:
            return 0
        return (s0 + self.n_steps) // self.record_every - s0 // self.record_every


def _rng(seed: int, tag: int) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(key=[seed & 0xFFFFFFFFFFFFFFFF, tag]))


def _attitude_cmds(rng, K, MN, rp, thrust_lo, thrust_hi) -> np.ndarray:
    c = np.zeros((K, MN, 4), dtype=np.float32)
    c[..., 0] = rng.uniform(-rp, rp, (K, MN))
    c[..., 1] = rng.uniform(-rp, rp, (K, MN))
    if thrust_lo == thrust_hi:
        c[..., 3] = thrust_lo
    else:
        c[..., 3] = rng.uniform(thrust_lo, thrust_hi, (K, MN))
    return c


def cfg1(seed=REPORT_SEED, n_steps=1000, M=1) -> Workload:
    """configs[0]: single drone, FP, Euler 1000 Hz, attitude controller 500 Hz, record every step."""
    rng = _rng(seed, 1)
    cmds = _attitude_cmds(rng, 1, M, 0.2, 0.265, 0.265)
    return Workload("cfg1", M, 1, MODEL_FP,
                    dict(integrator=EULER, iface=IF_ATTITUDE, f_phys=1000.0, f_att=500.0, init_mode=0),
                    seed, n_steps, n_steps, 1, cmds)


def cfg2(seed=REPORT_SEED, M=4096, n_steps=2000) -> Workload:
    """configs[1]: 4096 worlds, FP, RK4 1000 Hz, attitude commands redrawn every 50 steps, record every 10th."""
    rng = _rng(seed, 2)
    hold = 50
    K = -(-n_steps // hold)
    cmds = _attitude_cmds(rng, K, M, 0.3, 0.15, 0.40)
    return Workload("cfg2", M, 1, MODEL_FP,
                    dict(integrator=RK4, iface=IF_ATTITUDE, f_phys=1000.0, f_att=500.0, init_mode=1,
                         p0_lo=[-1, -1, 0], p0_hi=[1, 1, 2], tilt0_max=0.5),
                    seed, n_steps, hold, 10, cmds)


def _obstacles(seed) -> np.ndarray:
    rng = _rng(seed, 30)
    o = np.zeros((8, 4))
    o[:, 0] = rng.uniform(0.5, 3.0, 8)
    o[:, 1] = rng.uniform(-1.5, 1.5, 8)
    o[:, 2] = rng.uniform(0.3, 1.7, 8)
    o[:, 3] = rng.uniform(0.1, 0.3, 8)
    return o.astype(np.float32).astype(np.float64)   # exactly representable in float32 on both sides


_CFG3_SIGMA = [0.15, 0.15, 0.05, 0.03]
_CFG3_LO = [-0.5, -0.5, -math.pi, 0.05]
_CFG3_HI = [0.5, 0.5, math.pi, 0.55]


def _cfg3_params(seed):
    lo, hi = [1.0] * 12, [1.0] * 12
    for s in (1, 2, 3, 4, 5, 6, 8, 9, 10):           # a[3], b[3], c[3] of Eq. (10), +-10 % per world and axis
        lo[s], hi[s] = 0.9, 1.1
    return dict(integrator=EULER, iface=IF_ATTITUDE, f_phys=500.0, f_att=500.0, init_mode=0,
                rnd_lo=lo, rnd_hi=hi, n_obstacles=8, obstacles=_obstacles(seed),
                noise_sigma=_CFG3_SIGMA, cmd_lo=_CFG3_LO, cmd_hi=_CFG3_HI)


def _cfg3_start() -> np.ndarray:
    x = np.zeros(13)
    x[2] = 1.0
    x[6] = 1.0
    x[12] = np.float32(MASS * G)
    return x


def cfg3(seed=REPORT_SEED, M=1 << 20, n_steps=100) -> Workload:
    """configs[2]: 2^20 rollouts, AB model, in-kernel nominal+noise commands, fused, final state + min distance."""
    nominal = np.zeros((n_steps, 4), dtype=np.float32)
    nominal[:, 3] = MASS * G
    p = _cfg3_params(seed)
    p["cmd_source"] = CMD_NOMINAL_PLUS_NOISE
    return Workload("cfg3", M, 1, MODEL_AB, p, seed, n_steps, 1, 0, nominal, broadcast_state=_cfg3_start())


def cfg3b(seed=REPORT_SEED, M=1 << 20, n_steps=100, host_cmds=True) -> Workload:
    """Variant 3B: the same rollout with the command sequences supplied as a [K][M] float4 buffer."""
    cmds = None
    if host_cmds:
        rng = _rng(seed, 31)
        cmds = np.zeros((n_steps, M, 4), dtype=np.float32)
        nominal = np.array([0, 0, 0, MASS * G])
        for j in range(4):
            cmds[..., j] = np.clip(nominal[j] + _CFG3_SIGMA[j] * rng.standard_normal((n_steps, M), dtype=np.float32),
                                   _CFG3_LO[j], _CFG3_HI[j])
    p = _cfg3_params(seed)
    p["cmd_source"] = CMD_BUFFER
    return Workload("cfg3b", M, 1, MODEL_AB, p, seed, n_steps, 1, 0, cmds, broadcast_state=_cfg3_start(),
                    notes=dict(sigma=_CFG3_SIGMA, lo=_CFG3_LO, hi=_CFG3_HI, nominal=[0, 0, 0, MASS * G]))


def cfg4(seed=REPORT_SEED, M=1000, N=4000, n_steps=500) -> Workload:
    """configs[3]: swarms of N drones on a 16^3 grid, AB model, position interface at 100 Hz, per-world mass."""
    rng = _rng(seed, 4)
    spacing, origin = 0.3, np.array([-2.25, -2.25, 0.5])
    n = np.arange(N)
    cell = np.stack([n % 16, (n // 16) % 16, n // 256], axis=1)
    p0 = origin + spacing * cell                                  # grid cell centres (layout, not physics)
    cmds = np.zeros((1, M * N, 4), dtype=np.float32)
    tgt = np.tile(p0, (M, 1)) + rng.uniform(-0.5, 0.5, (M * N, 3))
    cmds[0, :, :3] = tgt
    lo, hi = [1.0] * 12, [1.0] * 12
    lo[0], hi[0] = 0.025 / MASS, 0.032 / MASS
    gz = max(1, -(-N // 256))
    return Workload("cfg4", M, N, MODEL_AB,
                    dict(integrator=EULER, iface=IF_POSITION, f_phys=500.0, f_att=500.0, f_pos=100.0,
                         init_mode=2, grid_dims=[16, 16, max(16, gz)], grid_spacing=spacing, grid_jitter=0.02,
                         grid_origin=origin.tolist(), rnd_lo=lo, rnd_hi=hi),
                    seed, n_steps, n_steps, 50, cmds)


def cfg5(seed=REPORT_SEED, M=65536, n_steps=1000, integrator=RK4) -> Workload:
    """configs[4]: domain randomisation + Philox force disturbances, RK4 1000 Hz, record every step."""
    rng = _rng(seed, 5)
    cmds = _attitude_cmds(rng, 1, M, 0.2, 0.265, 0.265)
    lo, hi = [1.0] * 12, [1.0] * 12
    for s in (0, 1, 2, 3):
        lo[s], hi[s] = 0.9, 1.1                                   # mass, Jx, Jy, Jz
    lo[4], hi[4] = 0.95, 1.05                                     # k_f
    return Workload("cfg5" if integrator == RK4 else "cfg5e", M, 1, MODEL_FP,
                    dict(integrator=integrator, iface=IF_ATTITUDE, f_phys=1000.0, f_att=500.0, init_mode=0,
                         rnd_lo=lo, rnd_hi=hi, dist_sigma=0.005),
                    seed, n_steps, n_steps, 1, cmds)


def cfg5e(seed=REPORT_SEED, M=65536, n_steps=1000) -> Workload:
    """Variant 5E: as configs[4] with explicit Euler -- the unambiguously memory-bound record mode."""
    return cfg5(seed, M, n_steps, integrator=EULER)


def mppi(seed=REPORT_SEED, n_ctrl=5, worlds_per_ctrl=100_000, horizon=25, cmd_hold=10, n_elite=None) -> Workload:
    """The sampling-based planner of PAPER.md:L465-L471 around the configs[2] rollout: 5 controllers x 100 000 rollouts
    (500 k), 25 knots at 50 Hz (10 physics steps of the 500 Hz abstracted model per knot), top 1 % elites, AR(1) noise.
    The paper's own parameters are in a codebase that is not available; the values here are this build's choice."""
    p = _cfg3_params(seed)
    p.update(cmd_source=CMD_NOMINAL_PLUS_NOISE, noise_beta=0.7, n_ctrl=n_ctrl, worlds_per_ctrl=worlds_per_ctrl,
             cost_on=1, cost_goal=[3.5, 0.0, 1.0], cost_w_pos=1.0, cost_w_vel=0.05, cost_w_term=10.0,
             cost_w_obs=200.0, cost_d_safe=0.15, cost_w_coll=1000.0)
    nominal = np.zeros((n_ctrl, horizon, 4), dtype=np.float32)
    nominal[..., 3] = MASS * G
    if n_elite is None:
        n_elite = max(1, worlds_per_ctrl // 100)
    return Workload("mppi", n_ctrl * worlds_per_ctrl, 1, MODEL_AB, p, seed, horizon * cmd_hold, cmd_hold, 0, nominal,
                    broadcast_state=_cfg3_start(),
                    notes=dict(horizon=horizon, n_elite=n_elite, lam=0.5, shift=1, n_ctrl=n_ctrl))


def grad(seed=REPORT_SEED, M=1 << 20, n_steps=10, host_cmds=True) -> Workload:
    """Fig. 3D: 2^20 worlds, first-principles model + attitude controller, RK4, the goal distance
    after 10 steps differentiated w.r.t. the 10 attitude commands."""
    cmds = _attitude_cmds(_rng(seed, 6), n_steps, M, 0.2, 0.2, 0.35) if host_cmds else None
    return Workload("grad", M, 1, MODEL_FP,
                    dict(integrator=RK4, iface=IF_ATTITUDE, f_phys=1000.0, f_att=500.0, init_mode=1,
                         p0_lo=[-1, -1, 0], p0_hi=[1, 1, 2], tilt0_max=0.4),
                    seed, n_steps, 1, 0, cmds, notes=dict(goal=[0.5, -0.2, 1.2]))


def depth(seed=REPORT_SEED, M=1024, model=MODEL_FP, width=64, height=64) -> Workload:
    """depth images, 64 x 64 rays x 1024 environments.  The paper's MuJoCo test scene is not available: a
    synthetic room of 16 spheres, 16 axis-aligned boxes and the ground plane stands in for it; every environment's drone
    hovers at a random pose (position box + tilt <= 0.4 rad), its camera looks along body +x."""
    rng = _rng(seed, 7)
    sph = np.column_stack([rng.uniform(2.0, 7.0, 16), rng.uniform(-3.0, 3.0, 16), rng.uniform(0.3, 2.5, 16),
                           rng.uniform(0.15, 0.6, 16)])
    box = np.column_stack([rng.uniform(2.0, 8.0, 16), rng.uniform(-3.5, 3.5, 16), rng.uniform(0.2, 2.0, 16),
                           rng.uniform(0.1, 0.5, (16, 3))])
    scene = dict(width=width, height=height, fov_x=1.2, spheres=sph.astype(np.float32).astype(np.float64),
                 boxes=box.astype(np.float32).astype(np.float64), ground_plane=True, cam_offset=(0.03, 0.0, 0.0), t_max=20.0)
    fp = model == MODEL_FP
    return Workload("depth", M, 1, model,
                    dict(integrator=EULER, iface=IF_ATTITUDE, f_phys=1000.0 if fp else 500.0, f_att=500.0, init_mode=1,
                         p0_lo=[-1, -1, 0.5], p0_hi=[1, 1, 2], tilt0_max=0.4),
                    seed, 1, 1, 0, None, notes=dict(scene=scene))


# ---- round 3: configurations of the paper's tasks that are NOT BASELINE.json benchmark rows ----
def fp_pos(seed=REPORT_SEED, M=1 << 16, n_steps=500) -> Workload:
    """The full onboard stack on the first-principles model: position targets -> geometric position controller (100 Hz)
    -> attitude controller + mixer (500 Hz) -> Eqs. (1)-(6), RK4 1000 Hz; nominal plant, nothing recorded."""
    rng = _rng(seed, 11)
    cmds = np.zeros((1, M, 4), dtype=np.float32)
    cmds[0, :, :3] = rng.uniform([-1, -1, 0.5], [1, 1, 1.5], (M, 3))
    cmds[0, :, 3] = rng.uniform(-0.5, 0.5, M)
    return Workload("fp_pos", M, 1, MODEL_FP,
                    dict(integrator=RK4, iface=IF_POSITION, f_phys=1000.0, f_att=500.0, f_pos=100.0, init_mode=1,
                         p0_lo=[-1, -1, 0.5], p0_hi=[1, 1, 1.5], tilt0_max=0.3),
                    seed, n_steps, n_steps, 0, cmds)


def fp_rotor(seed=REPORT_SEED, M=1 << 20, n_steps=100) -> Workload:
    """Motor-level control ("direct rotor velocity"): four rotor speed commands per drone, redrawn every 50
    steps; first-principles model, RK4 1000 Hz, nominal plant, nothing recorded."""
    rng = _rng(seed, 12)
    hold = 50
    cmds = rng.uniform(12000.0, 17000.0, (-(-n_steps // hold), M, 4)).astype(np.float32)
    return Workload("fp_rotor", M, 1, MODEL_FP,
                    dict(integrator=RK4, iface=IF_ROTOR, f_phys=1000.0, f_att=500.0, init_mode=1, p0_lo=[-1, -1, 0],
                         p0_hi=[1, 1, 2], tilt0_max=0.5),
                    seed, n_steps, hold, 0, cmds)


def ab_rk4(seed=REPORT_SEED, M=1 << 20, n_steps=100) -> Workload:
    """The abstracted model integrated with RK4 (the paper's benchmark rows use Euler for it): attitude commands redrawn
    every 50 steps, 500 Hz, nothing recorded.  Runs the general kernel (no lean instantiation)."""
    rng = _rng(seed, 13)
    hold = 50
    cmds = _attitude_cmds(rng, -(-n_steps // hold), M, 0.3, 0.2, 0.33)
    return Workload("ab_rk4", M, 1, MODEL_AB,
                    dict(integrator=RK4, iface=IF_ATTITUDE, f_phys=500.0, f_att=500.0, init_mode=1, p0_lo=[-1, -1, 0],
                         p0_hi=[1, 1, 2], tilt0_max=0.4),
                    seed, n_steps, hold, 0, cmds)


REGISTRY = {"fp_pos": fp_pos, "fp_rotor": fp_rotor, "ab_rk4": ab_rk4, "depth": depth, "grad": grad, "mppi": mppi, "cfg1": cfg1, "cfg2": cfg2, "cfg3": cfg3, "cfg3b": cfg3b, "cfg4": cfg4, "cfg5": cfg5, "cfg5e": cfg5e}


def make(name: str, **kw) -> Workload:
    return REGISTRY[name](**kw)


def shard_worlds(M: int, world_size: int, rank: int) -> tuple[int, int]:
    """Contiguous partition of the world axis: returns (world_offset, local M)."""
    base, rem = divmod(M, world_size)
    lo = rank * base + min(rank, rem)
    return lo, base + (1 if rank < rem else 0)
