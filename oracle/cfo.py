"""ctypes binding of the float64 CPU ORACLE (oracle/cfo.c).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs.  Never imported by the product package
paper_2606_01478_b200, and never imports it.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libcfo.so")
_SRC = [os.path.join(_HERE, "cfo.c"), os.path.join(_HERE, "cfo.h")]

MODEL_FP, MODEL_AB = 0, 1
EULER, RK4 = 0, 1
IF_ROTOR, IF_TORQUE, IF_ATTITUDE, IF_POSITION = 0, 1, 2, 3
CMD_BUFFER, CMD_NOMINAL_PLUS_NOISE = 0, 1
AUX_COUNTERS, AUX_MIN_DIST, AUX_CTRL, AUX_WORLD_PARAMS, AUX_REC_TABLE, AUX_MIN_D2, AUX_COST, AUX_EPS, AUX_COST_RUN = range(9)
REC_TABLE_CAP = 4096

d = C.c_double


class Params(C.Structure):
    _fields_ = [
        ("integrator", C.c_int32), ("iface", C.c_int32), ("cmd_source", C.c_int32), ("ab_thrust_dyn", C.c_int32),
        ("init_mode", C.c_int32), ("grid_dims", C.c_int32 * 3), ("n_obstacles", C.c_int32), ("_pad", C.c_int32),
        ("world_offset", C.c_int64),
        ("f_phys", d), ("f_att", d), ("f_pos", d),
        ("mass", d), ("J", d * 3), ("arm", d), ("kf", d * 3), ("km", d * 3), ("g", d),
        ("cv_up", d), ("cv_dn", d), ("cd_up", d), ("cd_dn", d),
        ("Jp", d), ("Ca", d * 3),
        ("ab_a", d * 3), ("ab_b", d * 3), ("ab_c", d * 3), ("ab_ctau", d), ("ab_cf", d),
        ("rpm_min", d), ("rpm_max", d), ("thrust_min", d), ("thrust_max", d), ("tilt_max", d),
        ("kR", d * 3), ("kW", d * 3), ("kI", d * 3), ("iR_max", d),
        ("kp", d * 3), ("kd", d * 3), ("ki", d * 3), ("ip_max", d * 3),
        ("rnd_lo", d * 12), ("rnd_hi", d * 12),
        ("dist_sigma", d),
        ("p0_lo", d * 3), ("p0_hi", d * 3), ("tilt0_max", d),
        ("grid_spacing", d), ("grid_jitter", d), ("grid_origin", d * 3),
        ("obstacles", (d * 4) * 8),
        ("noise_sigma", d * 4), ("cmd_lo", d * 4), ("cmd_hi", d * 4),
        ("noise_beta", d), ("worlds_per_ctrl", C.c_int64), ("n_ctrl", C.c_int32), ("cost_on", C.c_int32),
        ("cost_goal", d * 3), ("cost_w_pos", d), ("cost_w_vel", d), ("cost_w_term", d), ("cost_w_obs", d),
        ("cost_d_safe", d), ("cost_w_coll", d),
    ]


def build(force: bool = False) -> str:
    """Compile oracle/cfo.c -> oracle/libcfo.so (gcc -O2, no fast-math, OpenMP over drones)."""
    if not force and os.path.exists(_LIB_PATH) and all(
            os.path.getmtime(_LIB_PATH) >= os.path.getmtime(s) for s in _SRC):
        return _LIB_PATH
    cmd = ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
           "-o", _LIB_PATH, _SRC[0], "-lm"]
    subprocess.run(cmd, check=True, cwd=_HERE)
    return _LIB_PATH


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB_PATH)
        vp = C.c_void_p
        L.cfo_default_params.argtypes = [C.POINTER(Params), C.c_int]
        L.cfo_default_params.restype = None
        L.cfo_create.argtypes = [C.POINTER(vp), C.c_int64, C.c_int64, C.c_int, C.POINTER(Params)]
        L.cfo_destroy.argtypes = [vp]
        L.cfo_destroy.restype = None
        L.cfo_reset.argtypes = [vp, C.c_uint64]
        L.cfo_set_state.argtypes = [vp, vp, C.c_int]
        L.cfo_reset_masked.argtypes = [vp, vp, C.c_uint64]
        L.cfo_set_full.argtypes = [vp, vp, vp, vp, vp, C.c_int64]
        L.cfo_set_plan_state.argtypes = [vp, vp, vp]
        L.cfo_step.argtypes = [vp, vp, C.c_int, C.c_int, C.c_int, C.c_int, vp, C.c_size_t]
        L.cfo_step_f64cmd.argtypes = [vp, vp, C.c_int, C.c_int, C.c_int]
        L.cfo_get_state.argtypes = [vp, vp]
        L.cfo_get_aux.argtypes = [vp, C.c_int, vp]
        L.cfo_philox.argtypes = [C.c_uint64, C.POINTER(C.c_uint32 * 4), C.POINTER(C.c_uint32 * 4)]
        L.cfo_philox.restype = None
        L.cfo_uniform.argtypes = [C.c_uint32]
        L.cfo_uniform.restype = d
        L.cfo_normal_pair.argtypes = [C.c_uint32, C.c_uint32, C.POINTER(d), C.POINTER(d)]
        L.cfo_normal_pair.restype = None
        L.cfo_attitude_tick.argtypes = [C.POINTER(Params)] + [vp] * 7
        L.cfo_attitude_tick.restype = None
        L.cfo_position_tick.argtypes = [C.POINTER(Params)] + [vp] * 6
        L.cfo_position_tick.restype = None
        L.cfo_mix.argtypes = [C.POINTER(Params), vp, C.POINTER(d), vp]
        L.cfo_mix.restype = None
        L.cfo_num_threads.restype = C.c_int
        L.cfo_set_num_threads.argtypes = [C.c_int]
        L.cfo_set_num_threads.restype = None
        _lib = L
    return _lib


def _assign(struct, key, val):
    cur = getattr(struct, key)
    if not isinstance(cur, C.Array):
        setattr(struct, key, val)
        return
    flat = np.asarray(val).reshape(-1).tolist()
    if isinstance(cur[0], C.Array):          # 2-D (obstacles[8][4]); fewer rows than 8 allowed
        inner = len(cur[0])
        if len(flat) % inner or len(flat) > inner * len(cur):
            raise ValueError(f"{key}: bad size {len(flat)}")
        for r in range(len(flat) // inner):
            for c_ in range(inner):
                cur[r][c_] = flat[r * inner + c_]
    else:
        if len(flat) != len(cur):
            raise ValueError(f"{key}: expected {len(cur)} values, got {len(flat)}")
        for j, v in enumerate(flat):
            cur[j] = v


def make_params(model: int, overrides: dict | None = None) -> Params:
    p = Params()
    lib().cfo_default_params(C.byref(p), model)
    for k, v in (overrides or {}).items():
        _assign(p, k, v)
    return p


def _ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _f64(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


class OracleSim:
    """Same call names as the product binding (create/reset/step/get_state), float64 numpy in and out."""

    def __init__(self, M: int, N: int, model: int, overrides: dict | None = None):
        self.M, self.N, self.model = int(M), int(N), int(model)
        self.MN = self.M * self.N
        self.D = 17 if model == MODEL_FP else 13
        self.P = 14 if model == MODEL_FP else 11
        self.params = make_params(model, overrides)
        self._h = C.c_void_p()
        rc = lib().cfo_create(C.byref(self._h), self.M, self.N, model, C.byref(self.params))
        if rc != 0:
            raise ValueError(f"cfo_create failed: {rc}")

    def __del__(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            lib().cfo_destroy(self._h)
            self._h = C.c_void_p()

    def reset(self, seed: int):
        rc = lib().cfo_reset(self._h, seed)
        assert rc == 0, rc

    def reset_masked(self, mask, episode_seed: int):
        m = np.ascontiguousarray(mask, dtype=np.uint8)
        assert m.size == self.M
        rc = lib().cfo_reset_masked(self._h, _ptr(m), int(episode_seed))
        assert rc == 0, rc

    def set_state(self, state, broadcast: bool = False):
        st = _f64(state)
        assert st.size == (self.D if broadcast else self.D * self.MN)
        rc = lib().cfo_set_state(self._h, _ptr(st), int(broadcast))
        if rc != 0:
            raise RuntimeError(f"cfo_set_state: {rc}")

    def set_full(self, state=None, ctrl=None, wparam=None, mind2=None, step_counter=-1):
        st, ct, wp, md = _f64(state), _f64(ctrl), _f64(wparam), _f64(mind2)
        for a, n in ((st, self.D * self.MN), (ct, 14 * self.MN), (wp, self.P * self.M), (md, 8 * self.MN)):
            assert a is None or a.size == n
        rc = lib().cfo_set_full(self._h, _ptr(st), _ptr(ct), _ptr(wp), _ptr(md), int(step_counter))
        assert rc == 0, rc

    def n_records(self, n_steps: int, record_every: int) -> int:
        if record_every <= 0:
            return 0
        s0 = int(self.counters()[0])
        return (s0 + n_steps) // record_every - s0 // record_every

    def step(self, cmds, n_steps: int, cmd_hold: int = 1, record_every: int = 0, check: bool = True):
        """cmds: float32 [K][M*N][4] (buffer source) or [n_ctrl][K][4] (nominal + noise).  Returns record
        [n_rec][D][M*N] float64 (or None)."""
        cm = np.ascontiguousarray(cmds, dtype=np.float32)
        per = 4 * self.MN if self.params.cmd_source == CMD_BUFFER else 4 * self.params.n_ctrl
        assert cm.size % per == 0, (cm.shape, per)
        n_cmds = cm.size // per
        n_rec = self.n_records(n_steps, record_every)
        rec = np.empty((n_rec, self.D, self.MN), dtype=np.float64) if n_rec else None
        rc = lib().cfo_step(self._h, _ptr(cm), n_cmds, cmd_hold, n_steps, record_every,
                            _ptr(rec), 0 if rec is None else rec.size)
        if check and rc != 0:
            raise RuntimeError(f"cfo_step: {rc}")
        return rec if check else (rc, rec)

    def step_f64(self, cmds64, n_steps: int, cmd_hold: int = 1):
        """cmds64: float64 [K][M*N][4], command-buffer source only (oracle/grad.py)."""
        cm = np.ascontiguousarray(cmds64, dtype=np.float64)
        assert cm.size % (4 * self.MN) == 0
        rc = lib().cfo_step_f64cmd(self._h, _ptr(cm), cm.size // (4 * self.MN), cmd_hold, n_steps)
        if rc != 0:
            raise RuntimeError(f"cfo_step_f64cmd: {rc}")

    def get_state(self):
        out = np.empty((self.D, self.MN), dtype=np.float64)
        assert lib().cfo_get_state(self._h, _ptr(out)) == 0
        return out

    def counters(self):
        out = np.zeros(4, dtype=np.uint32)
        assert lib().cfo_get_aux(self._h, AUX_COUNTERS, _ptr(out)) == 0
        return out

    def min_dist(self):
        out = np.empty(self.M, dtype=np.float64)
        assert lib().cfo_get_aux(self._h, AUX_MIN_DIST, _ptr(out)) == 0
        return out

    def ctrl(self):
        out = np.empty((14, self.MN), dtype=np.float64)
        assert lib().cfo_get_aux(self._h, AUX_CTRL, _ptr(out)) == 0
        return out

    def world_params(self):
        out = np.empty((self.P, self.M), dtype=np.float64)
        assert lib().cfo_get_aux(self._h, AUX_WORLD_PARAMS, _ptr(out)) == 0
        return out

    def min_d2(self):
        out = np.empty((8, self.MN), dtype=np.float64)
        assert lib().cfo_get_aux(self._h, AUX_MIN_D2, _ptr(out)) == 0
        return out

    def cost(self):
        out = np.empty(self.MN, dtype=np.float64)
        assert lib().cfo_get_aux(self._h, AUX_COST, _ptr(out)) == 0
        return out

    def cost_run(self):
        out = np.empty(self.MN, dtype=np.float64)
        assert lib().cfo_get_aux(self._h, AUX_COST_RUN, _ptr(out)) == 0
        return out

    def eps(self):
        out = np.empty((4, self.MN), dtype=np.float64)
        assert lib().cfo_get_aux(self._h, AUX_EPS, _ptr(out)) == 0
        return out

    def set_plan_state(self, eps=None, cost_run=None):
        e, c = _f64(eps), _f64(cost_run)
        assert e is None or e.size == 4 * self.MN
        assert c is None or c.size == self.MN
        assert lib().cfo_set_plan_state(self._h, _ptr(e), _ptr(c)) == 0

    def rec_table(self):
        out = np.zeros(REC_TABLE_CAP, dtype=np.uint32)
        assert lib().cfo_get_aux(self._h, AUX_REC_TABLE, _ptr(out)) == 0
        return out


def philox(seed: int, ctr) -> np.ndarray:
    c = (C.c_uint32 * 4)(*[int(v) for v in ctr])
    o = (C.c_uint32 * 4)()
    lib().cfo_philox(seed, C.byref(c), C.byref(o))
    return np.array(list(o), dtype=np.uint32)


def uniform(x: int) -> float:
    return lib().cfo_uniform(int(x))


def normal_pair(xa: int, xb: int):
    z0, z1 = d(), d()
    lib().cfo_normal_pair(int(xa), int(xb), C.byref(z0), C.byref(z1))
    return z0.value, z1.value


def attitude_tick(params: Params, q, w, cmd, iR):
    q, w, cmd = _f64(q), _f64(w), _f64(cmd)
    iR = np.array(iR, dtype=np.float64)
    eR, tau, rpm = np.zeros(3), np.zeros(3), np.zeros(4)
    lib().cfo_attitude_tick(C.byref(params), _ptr(q), _ptr(w), _ptr(cmd), _ptr(iR), _ptr(eR), _ptr(tau), _ptr(rpm))
    return eR, iR, tau, rpm


def position_tick(params: Params, pos, vel, zB, target, ip):
    pos, vel, zB, target = _f64(pos), _f64(vel), _f64(zB), _f64(target)
    ip = np.array(ip, dtype=np.float64)
    att = np.zeros(4)
    lib().cfo_position_tick(C.byref(params), _ptr(pos), _ptr(vel), _ptr(zB), _ptr(target), _ptr(ip), _ptr(att))
    return att, ip


def mix(params: Params, rpm):
    rpm = _f64(rpm)
    F = d()
    tau = np.zeros(3)
    lib().cfo_mix(C.byref(params), _ptr(rpm), C.byref(F), _ptr(tau))
    return F.value, tau


def num_threads() -> int:
    return lib().cfo_num_threads()


def set_num_threads(n: int):
    lib().cfo_set_num_threads(int(n))
