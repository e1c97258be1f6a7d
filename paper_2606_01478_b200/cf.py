"""Thin Python binding of libcf.so (include/cf.h): argument marshalling only.

PyTorch is used for device memory (`torch.empty`) and the current CUDA stream; every step of the path runs in the
library's own kernels.  There is no fallback: if libcf.so is missing this module raises on first use.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("CF_LIB") or os.path.join(_HERE, "libcf.so")    # CF_LIB: an alternative build (debug, variant)

MODEL_FP, MODEL_AB = 0, 1
EULER, RK4 = 0, 1
IF_ROTOR, IF_TORQUE, IF_ATTITUDE, IF_POSITION = 0, 1, 2, 3
CMD_BUFFER, CMD_NOMINAL_PLUS_NOISE = 0, 1
AUX_COUNTERS, AUX_MIN_DIST, AUX_CTRL, AUX_WORLD_PARAMS, AUX_REC_TABLE, AUX_MIN_D2, AUX_COST, AUX_EPS, AUX_COST_RUN, AUX_NONFINITE = range(10)
REC_TABLE_CAP = 4096
OK, E_ARG, E_SHAPE, E_STATE, E_BUFFER, E_CUDA, E_UNSUPPORTED = 0, -1, -2, -3, -4, -5, -6

f = C.c_float


class Params(C.Structure):
    """Mirror of `cf_params` (include/cf.h)."""
    _fields_ = [
        ("struct_size", C.c_uint32),
        ("integrator", C.c_int32), ("iface", C.c_int32), ("cmd_source", C.c_int32),
        ("ab_thrust_dyn", C.c_int32), ("init_mode", C.c_int32), ("grid_dims", C.c_int32 * 3),
        ("n_obstacles", C.c_int32), ("world_offset", C.c_int64),
        ("f_phys", f), ("f_att", f), ("f_pos", f),
        ("mass", f), ("J", f * 3), ("arm", f), ("kf", f * 3), ("km", f * 3), ("g", f),
        ("cv_up", f), ("cv_dn", f), ("cd_up", f), ("cd_dn", f),
        ("Jp", f), ("Ca", f * 3),
        ("ab_a", f * 3), ("ab_b", f * 3), ("ab_c", f * 3), ("ab_ctau", f), ("ab_cf", f),
        ("rpm_min", f), ("rpm_max", f), ("thrust_min", f), ("thrust_max", f), ("tilt_max", f),
        ("kR", f * 3), ("kW", f * 3), ("kI", f * 3), ("iR_max", f),
        ("kp", f * 3), ("kd", f * 3), ("ki", f * 3), ("ip_max", f * 3),
        ("rnd_lo", f * 12), ("rnd_hi", f * 12),
        ("dist_sigma", f),
        ("p0_lo", f * 3), ("p0_hi", f * 3), ("tilt0_max", f),
        ("grid_spacing", f), ("grid_jitter", f), ("grid_origin", f * 3),
        ("obstacles", (f * 4) * 8),
        ("noise_sigma", f * 4), ("cmd_lo", f * 4), ("cmd_hi", f * 4),
        ("noise_beta", f), ("n_ctrl", C.c_int32), ("worlds_per_ctrl", C.c_int64), ("cost_on", C.c_int32),
        ("cost_goal", f * 3), ("cost_w_pos", f), ("cost_w_vel", f), ("cost_w_term", f), ("cost_w_obs", f),
        ("cost_d_safe", f), ("cost_w_coll", f),
    ]


class MppiParams(C.Structure):
    """Mirror of `cf_mppi_params` (include/cf.h)."""
    _fields_ = [("struct_size", C.c_uint32), ("horizon", C.c_int32), ("cmd_hold", C.c_int32), ("n_elite", C.c_int32),
                ("shift", C.c_int32), ("lam", f)]


DEPTH_MAX_PRIMS = 32


class DepthParams(C.Structure):
    """Mirror of `cf_depth_params` (include/cf.h)."""
    _fields_ = [("struct_size", C.c_uint32), ("width", C.c_int32), ("height", C.c_int32), ("n_spheres", C.c_int32),
                ("n_boxes", C.c_int32), ("ground_plane", C.c_int32), ("fov_x", f), ("t_max", f), ("cam_offset", f * 3),
                ("spheres", (f * 4) * DEPTH_MAX_PRIMS), ("boxes", (f * 6) * DEPTH_MAX_PRIMS)]


class CfError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"cf status {code}: {msg}")
        self.code = code


_lib = None


def lib():
    """Load libcf.so (fails loudly if it was not built: there is no CPU path)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2606_01478_b200.build` "
                          "(or __graft_entry__.build()); this package has no CPU fallback")
    L = C.CDLL(LIB_PATH)
    vp, i64, sz = C.c_void_p, C.c_int64, C.c_size_t
    sig = {
        "cf_default_params": (None, [C.POINTER(Params), C.c_int]),
        "cf_state_dim": (C.c_int, [C.c_int]),
        "cf_world_param_dim": (C.c_int, [C.c_int]),
        "cf_workspace_bytes": (sz, [i64, i64, C.c_int, C.POINTER(Params)]),
        "cf_create": (C.c_int, [C.POINTER(vp), i64, i64, C.c_int, C.POINTER(Params), vp, sz]),
        "cf_destroy": (C.c_int, [vp]),
        "cf_set_stream": (C.c_int, [vp, vp]),
        "cf_reset": (C.c_int, [vp, C.c_uint64]),
        "cf_set_state": (C.c_int, [vp, vp, C.c_int]),
        "cf_reset_masked": (C.c_int, [vp, vp, C.c_uint64]),
        "cf_set_full": (C.c_int, [vp, vp, vp, vp, vp, i64]),
        "cf_step": (C.c_int, [vp, vp, C.c_int, C.c_int, C.c_int, C.c_int, vp, sz]),
        "cf_staging_bytes": (sz, [vp, C.c_int, C.c_int, C.c_int]),
        "cf_step_host": (C.c_int, [vp, vp, C.c_int, C.c_int, C.c_int, C.c_int, vp, sz, vp, sz]),
        "cf_rollout_host": (C.c_int, [vp, vp, vp, C.c_int, C.c_int, C.c_int, vp, vp, vp, sz, C.c_int]),
        "cf_get_state": (C.c_int, [vp, vp]),
        "cf_get_state_host": (C.c_int, [vp, vp]),
        "cf_get_aux": (C.c_int, [vp, C.c_int, vp]),
        "cf_get_aux_host": (C.c_int, [vp, C.c_int, vp, vp, sz]),
        "cf_step_counter": (i64, [vp]),
        "cf_sync_counters": (C.c_int, [vp]),
        "cf_describe_launch": (C.c_int, [vp, C.c_char_p, sz, C.POINTER(C.c_int), C.POINTER(C.c_int)]),
        "cf_set_plan_state": (C.c_int, [vp, vp, vp]),
        "cf_mppi_scratch_bytes": (sz, [vp, C.POINTER(MppiParams)]),
        "cf_mppi_update": (C.c_int, [vp, C.POINTER(MppiParams), vp, vp, vp, vp, vp, sz]),
        "cf_set_counters": (C.c_int, [vp, C.POINTER(C.c_uint32 * 4), vp]),
        "cf_set_copy_stream": (C.c_int, [vp, vp]),
        "cf_mppi_update_static": (C.c_int, [vp, C.POINTER(MppiParams), vp, vp, vp, vp]),
        "cf_mppi_iterate": (C.c_int, [vp, C.POINTER(MppiParams), vp, vp, vp, vp, vp, vp, sz]),
        "cf_mppi_iterate_host": (C.c_int, [vp, C.POINTER(MppiParams), vp, vp, vp, vp, vp, vp, vp, sz]),
        "cf_mppi_pack_best": (C.c_int, [vp, C.POINTER(MppiParams), vp, vp, C.c_int, vp]),
        "cf_mppi_select": (C.c_int, [vp, vp, C.c_int, C.c_int, vp]),
        "cf_grad_scratch_bytes": (sz, [vp, C.c_int]),
        "cf_grad_staging_bytes": (sz, [vp, C.c_int]),
        "cf_grad_host": (C.c_int, [vp, vp, C.c_int, C.c_int, C.c_int, C.POINTER(C.c_float * 3), vp, vp, vp, sz, vp, sz]),
        "cf_depth_host": (C.c_int, [vp, C.POINTER(DepthParams), vp, vp, vp, sz]),
        "cf_grad": (C.c_int, [vp, vp, C.c_int, C.c_int, C.c_int, C.POINTER(C.c_float * 3), vp, vp, vp, sz]),
        "cf_depth": (C.c_int, [vp, C.POINTER(DepthParams), vp]),
        "cf_last_error": (C.c_char_p, []),
        "cf_debug_philox": (C.c_int, [C.c_uint64, C.POINTER(C.c_uint32 * 4), C.POINTER(C.c_uint32 * 4)]),
        "cf_debug_philox_dev": (C.c_int, [vp, C.c_uint64, vp, C.c_int, vp, vp, vp]),
    }
    for name, (res, args) in sig.items():
        fn = getattr(L, name)
        fn.restype, fn.argtypes = res, args
    _lib = L
    return L


EXPORTS = ["cf_default_params", "cf_state_dim", "cf_world_param_dim", "cf_workspace_bytes", "cf_create", "cf_destroy",
           "cf_set_stream", "cf_reset", "cf_set_state", "cf_set_full", "cf_step", "cf_staging_bytes", "cf_step_host",
           "cf_get_state", "cf_get_state_host", "cf_get_aux", "cf_get_aux_host", "cf_step_counter", "cf_sync_counters",
           "cf_describe_launch", "cf_last_error", "cf_debug_philox", "cf_debug_philox_dev", "cf_set_plan_state",
           "cf_mppi_scratch_bytes", "cf_mppi_update", "cf_mppi_iterate", "cf_mppi_iterate_host", "cf_grad_scratch_bytes",
           "cf_grad", "cf_depth", "cf_reset_masked", "cf_grad_staging_bytes", "cf_grad_host", "cf_depth_host",
           "cf_mppi_pack_best", "cf_mppi_select", "cf_rollout_host", "cf_mppi_update_static",
           "cf_set_counters", "cf_set_copy_stream"]


def _check(rc: int):
    if rc != 0:
        raise CfError(rc, lib().cf_last_error().decode())


def _assign(struct, key, val):
    cur = getattr(struct, key)
    if not isinstance(cur, C.Array):
        setattr(struct, key, val)
        return
    flat = np.asarray(val).reshape(-1).tolist()
    if isinstance(cur[0], C.Array):
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


def default_params(model: int, overrides: dict | None = None) -> Params:
    p = Params()
    lib().cf_default_params(C.byref(p), model)
    for k, v in (overrides or {}).items():
        _assign(p, k, v)
    return p


def debug_philox(seed: int, ctr) -> np.ndarray:
    c = (C.c_uint32 * 4)(*[int(v) for v in ctr])
    o = (C.c_uint32 * 4)()
    _check(lib().cf_debug_philox(seed, C.byref(c), C.byref(o)))
    return np.array(list(o), dtype=np.uint32)


def _torch():
    import torch
    return torch


def _dptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


class Sim:
    """cf_create / cf_reset / cf_step / cf_get_state with torch tensors as the caller-owned device buffers."""

    def __init__(self, M: int, N: int, model: int, overrides: dict | None = None, device="cuda:0"):
        torch = _torch()
        self.M, self.N, self.model = int(M), int(N), int(model)
        self.MN = self.M * self.N
        self.D = lib().cf_state_dim(model)
        self.P = lib().cf_world_param_dim(model)
        self.params = default_params(model, overrides)
        self.device = torch.device(device)
        nbytes = lib().cf_workspace_bytes(self.M, self.N, model, C.byref(self.params))
        self._h = C.c_void_p()
        if nbytes == 0:      # let cf_create report why
            _check(lib().cf_create(C.byref(self._h), self.M, self.N, model, C.byref(self.params), None, 0))
        self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        off = (-self.workspace.data_ptr()) % 256
        self._ws_ptr = self.workspace.data_ptr() + off
        _check(lib().cf_create(C.byref(self._h), self.M, self.N, model, C.byref(self.params),
                               C.c_void_p(self._ws_ptr), nbytes))
        self._staging = None
        self.bind_stream()

    def __del__(self):
        h = getattr(self, "_h", None)
        if h is not None and h.value and _lib is not None:
            _lib.cf_destroy(h)
            self._h = C.c_void_p()

    # -- plumbing ------------------------------------------------------------------------------------------------
    def bind_stream(self, stream=None):
        torch = _torch()
        st = stream if stream is not None else torch.cuda.current_stream(self.device)
        _check(lib().cf_set_stream(self._h, C.c_void_p(st.cuda_stream)))

    def _dev(self, a, dtype=None):
        torch = _torch()
        if isinstance(a, torch.Tensor):
            t = a.to(self.device)
            return t.contiguous() if dtype is None else t.to(dtype).contiguous()
        return torch.as_tensor(np.ascontiguousarray(a), device=self.device).to(dtype or torch.float32).contiguous()

    def describe_launch(self):
        buf = C.create_string_buffer(256)
        g, b = C.c_int(), C.c_int()
        _check(lib().cf_describe_launch(self._h, buf, 256, C.byref(g), C.byref(b)))
        return buf.value.decode(), g.value, b.value

    # -- the four calls ------------------------------------------------------------------------------------------
    def reset(self, seed: int):
        _check(lib().cf_reset(self._h, int(seed)))

    def reset_masked(self, mask, episode_seed: int):
        """mask: [M] (bool / uint8, host or device): worlds that start a new episode."""
        m = self._dev(np.asarray(mask, dtype=np.uint8) if not isinstance(mask, _torch().Tensor) else mask, _torch().uint8)
        assert m.numel() == self.M
        _check(lib().cf_reset_masked(self._h, _dptr(m), int(episode_seed)))

    def set_state(self, state, broadcast: bool = False):
        t = self._dev(state, _torch().float32)
        assert t.numel() == (self.D if broadcast else self.D * self.MN)
        _check(lib().cf_set_state(self._h, _dptr(t), int(broadcast)))

    def set_full(self, state=None, ctrl=None, wparam=None, min_d2=None, step_counter=-1):
        f32 = _torch().float32
        ts = [None if a is None else self._dev(a, f32) for a in (state, ctrl, wparam, min_d2)]
        for t, n in zip(ts, (self.D * self.MN, 14 * self.MN, self.P * self.M, 8 * self.MN)):
            assert t is None or t.numel() == n
        _check(lib().cf_set_full(self._h, *[_dptr(t) for t in ts], int(step_counter)))

    def n_records(self, n_steps: int, record_every: int) -> int:
        if record_every <= 0:
            return 0
        s0 = self.step_counter
        return (s0 + n_steps) // record_every - s0 // record_every

    def step(self, cmds, n_steps: int, cmd_hold: int = 1, record_every: int = 0, record=None):
        """cmds: device tensor float32 [K][MN][4] (or [n_ctrl][K][4] for nominal+noise).  Returns the record tensor
        [n_rec][D][MN] (allocated here unless `record` is given) or None.  Asynchronous on the bound stream."""
        torch = _torch()
        cm = self._dev(cmds, torch.float32)
        per = 4 * self.MN if self.params.cmd_source == CMD_BUFFER else 4 * self.params.n_ctrl
        assert cm.numel() % per == 0, (tuple(cm.shape), per)
        n_rec = self.n_records(n_steps, record_every)
        if n_rec and record is None:
            record = torch.empty((n_rec, self.D, self.MN), dtype=torch.float32, device=self.device)
        _check(lib().cf_step(self._h, _dptr(cm), cm.numel() // per, int(cmd_hold), int(n_steps), int(record_every),
                             _dptr(record) if n_rec else None, record.numel() * 4 if n_rec else 0))
        return record[:n_rec] if n_rec else None

    def get_state(self):
        out = _torch().empty((self.D, self.MN), dtype=_torch().float32, device=self.device)
        _check(lib().cf_get_state(self._h, _dptr(out)))
        return out

    # -- host-buffer (end-to-end) path ---------------------------------------------------------------------------
    def step_host(self, cmds_host, n_steps: int, cmd_hold: int = 1, record_every: int = 0, record_host=None):
        """cmds_host / record_host: CPU tensors (pinned for full speed).  Synchronous."""
        torch = _torch()
        per = 4 * self.MN if self.params.cmd_source == CMD_BUFFER else 4 * self.params.n_ctrl
        assert cmds_host.dtype == torch.float32 and cmds_host.is_contiguous() and not cmds_host.is_cuda
        n_cmds = cmds_host.numel() // per
        need = lib().cf_staging_bytes(self._h, n_cmds, int(n_steps), int(record_every))
        if self._staging is None or self._staging.numel() < need + 256:
            self._staging = torch.empty(need + 256, dtype=torch.uint8, device=self.device)
        sp = self._staging.data_ptr() + (-self._staging.data_ptr()) % 256
        n_rec = self.n_records(n_steps, record_every)
        if n_rec and record_host is None:
            record_host = torch.empty((n_rec, self.D, self.MN), dtype=torch.float32, pin_memory=True)
        _check(lib().cf_step_host(self._h, C.c_void_p(cmds_host.data_ptr()), n_cmds, int(cmd_hold), int(n_steps),
                                  int(record_every), C.c_void_p(record_host.data_ptr()) if n_rec else None,
                                  record_host.numel() * 4 if n_rec else 0, C.c_void_p(sp), need))
        return record_host[:n_rec] if n_rec else None

    def rollout_host(self, cmds_host, n_steps: int, state_host, cmd_hold: int = 1, x0_host=None, min_dist_host=None,
                     n_slices: int = 8):
        """cf_rollout_host: broadcast start (x0_host [D] or None), fused rollout, final state [D][MN] and minimum distance
        [MN] back in (pinned) CPU tensors, the copies overlapped with the kernel slice by slice.  Synchronous."""
        torch = _torch()
        per = 4 * self.MN if self.params.cmd_source == CMD_BUFFER else 4 * self.params.n_ctrl
        assert cmds_host.dtype == torch.float32 and cmds_host.is_contiguous() and not cmds_host.is_cuda
        n_cmds = cmds_host.numel() // per
        need = lib().cf_staging_bytes(self._h, n_cmds, int(n_steps), 0) + 256
        if self._staging is None or self._staging.numel() < need + 256:
            self._staging = torch.empty(need + 256, dtype=torch.uint8, device=self.device)
        sp = self._staging.data_ptr() + (-self._staging.data_ptr()) % 256
        _check(lib().cf_rollout_host(self._h, C.c_void_p(x0_host.data_ptr()) if x0_host is not None else None,
                                     C.c_void_p(cmds_host.data_ptr()), n_cmds, int(cmd_hold), int(n_steps),
                                     C.c_void_p(state_host.data_ptr()),
                                     C.c_void_p(min_dist_host.data_ptr()) if min_dist_host is not None else None,
                                     C.c_void_p(sp), need, int(n_slices)))
        return state_host, min_dist_host

    def get_state_host(self, out=None):
        torch = _torch()
        if out is None:
            out = torch.empty((self.D, self.MN), dtype=torch.float32, pin_memory=True)
        _check(lib().cf_get_state_host(self._h, C.c_void_p(out.data_ptr())))
        return out

    def min_dist_host(self, out=None):
        torch = _torch()
        if out is None:
            out = torch.empty(self.M, dtype=torch.float32, pin_memory=True)
        if getattr(self, "_md_scratch", None) is None:
            self._md_scratch = torch.empty(self.M, dtype=torch.float32, device=self.device)
        scratch = self._md_scratch
        _check(lib().cf_get_aux_host(self._h, AUX_MIN_DIST, C.c_void_p(out.data_ptr()), _dptr(scratch), self.M * 4))
        return out

    # -- auxiliary outputs ---------------------------------------------------------------------------------------
    def _aux(self, which, shape, dtype):
        out = _torch().empty(shape, dtype=dtype, device=self.device)
        _check(lib().cf_get_aux(self._h, which, _dptr(out)))
        return out

    def counters(self):
        return self._aux(AUX_COUNTERS, (4,), _torch().int32).cpu().numpy().view(np.uint32)

    def min_dist(self, out=None):
        if out is None:
            return self._aux(AUX_MIN_DIST, (self.M,), _torch().float32)
        _check(lib().cf_get_aux(self._h, AUX_MIN_DIST, _dptr(out)))
        return out

    def ctrl(self):
        return self._aux(AUX_CTRL, (14, self.MN), _torch().float32)

    def world_params(self):
        return self._aux(AUX_WORLD_PARAMS, (self.P, self.M), _torch().float32)

    def min_d2(self):
        return self._aux(AUX_MIN_D2, (8, self.MN), _torch().float32)

    def cost(self):
        return self._aux(AUX_COST, (self.MN,), _torch().float32)

    def cost_run(self):
        return self._aux(AUX_COST_RUN, (self.MN,), _torch().float32)

    def eps(self):
        return self._aux(AUX_EPS, (4, self.MN), _torch().float32)

    def set_plan_state(self, eps=None, cost_run=None):
        f32 = _torch().float32
        e = None if eps is None else self._dev(eps, f32)
        c = None if cost_run is None else self._dev(cost_run, f32)
        assert e is None or e.numel() == 4 * self.MN
        assert c is None or c.numel() == self.MN
        _check(lib().cf_set_plan_state(self._h, _dptr(e), _dptr(c)))

    # -- depth ray casting (cf_depth) ------------------------------------------------------------------------------
    def depth_params(self, width: int, height: int, fov_x: float, spheres=(), boxes=(), ground_plane=False,
                     cam_offset=(0.0, 0.0, 0.0), t_max=0.0) -> DepthParams:
        dp = DepthParams()
        dp.struct_size = C.sizeof(DepthParams)
        dp.width, dp.height, dp.fov_x, dp.t_max, dp.ground_plane = int(width), int(height), float(fov_x), float(t_max), int(ground_plane)
        sp = np.asarray(spheres, dtype=np.float32).reshape(-1, 4)
        bx = np.asarray(boxes, dtype=np.float32).reshape(-1, 6)
        dp.n_spheres, dp.n_boxes = len(sp), len(bx)
        if len(sp) > DEPTH_MAX_PRIMS or len(bx) > DEPTH_MAX_PRIMS:
            raise ValueError("too many primitives")
        for r, row in enumerate(sp):
            for c_, v in enumerate(row):
                dp.spheres[r][c_] = float(v)
        for r, row in enumerate(bx):
            for c_, v in enumerate(row):
                dp.boxes[r][c_] = float(v)
        for j in range(3):
            dp.cam_offset[j] = float(cam_offset[j])
        return dp

    def depth(self, dp: DepthParams, out=None):
        """Depth images [MN][H][W] (device tensor) of every drone's camera at the current state."""
        if out is None:
            out = _torch().empty((self.MN, dp.height, dp.width), dtype=_torch().float32, device=self.device)
        _check(lib().cf_depth(self._h, C.byref(dp), _dptr(out)))
        return out

    def depth_host(self, dp: DepthParams, out_host, state_host=None):
        """End-to-end rendering: state_host [D][MN] (pinned CPU tensor of poses, or None) in, out_host [MN][H][W] (pinned) out."""
        torch = _torch()
        n = self.MN * dp.height * dp.width
        if getattr(self, "_depth_stage", None) is None or self._depth_stage.numel() < n:
            self._depth_stage = torch.empty(n, dtype=torch.float32, device=self.device)
        sp = None if state_host is None else C.c_void_p(state_host.data_ptr())
        _check(lib().cf_depth_host(self._h, C.byref(dp), sp, C.c_void_p(out_host.data_ptr()), _dptr(self._depth_stage), 4 * n))
        return out_host

    # -- gradient of the goal distance w.r.t. the commands (cf_grad) --------------------------------------------------
    def grad(self, cmds, n_steps: int, goal, cmd_hold: int = 1, loss=None, grad=None):
        """cmds: float32 [K][MN][4] (device).  Returns (loss [MN], grad [K][MN][4]) device tensors; the simulator state
        is left unchanged."""
        torch = _torch()
        cm = self._dev(cmds, torch.float32)
        assert cm.numel() % (4 * self.MN) == 0
        K = cm.numel() // (4 * self.MN)
        need = lib().cf_grad_scratch_bytes(self._h, int(n_steps))
        if getattr(self, "_grad_scratch", None) is None or self._grad_scratch.numel() < need + 16:
            self._grad_scratch = torch.empty(need + 16, dtype=torch.uint8, device=self.device)
        sp = self._grad_scratch.data_ptr() + (-self._grad_scratch.data_ptr()) % 16
        if loss is None:
            loss = torch.empty(self.MN, dtype=torch.float32, device=self.device)
        if grad is None:
            grad = torch.empty((K, self.MN, 4), dtype=torch.float32, device=self.device)
        g3 = (C.c_float * 3)(*[float(v) for v in goal])
        _check(lib().cf_grad(self._h, _dptr(cm), K, int(cmd_hold), int(n_steps), C.byref(g3), _dptr(loss), _dptr(grad),
                             C.c_void_p(sp), need))
        return loss, grad

    def grad_host(self, cmds_host, n_steps: int, goal, loss_host, grad_host, cmd_hold: int = 1):
        """End-to-end gradient: cmds_host [K][MN][4], loss_host [MN], grad_host [K][MN][4] are (pinned) CPU tensors."""
        torch = _torch()
        K = cmds_host.numel() // (4 * self.MN)
        need = lib().cf_grad_scratch_bytes(self._h, int(n_steps))
        if getattr(self, "_grad_scratch", None) is None or self._grad_scratch.numel() < need + 16:
            self._grad_scratch = torch.empty(need + 16, dtype=torch.uint8, device=self.device)
        sp = self._grad_scratch.data_ptr() + (-self._grad_scratch.data_ptr()) % 16
        st = lib().cf_grad_staging_bytes(self._h, K)
        if getattr(self, "_grad_stage", None) is None or self._grad_stage.numel() < st + 256:
            self._grad_stage = torch.empty(st + 256, dtype=torch.uint8, device=self.device)
        stp = self._grad_stage.data_ptr() + (-self._grad_stage.data_ptr()) % 256
        g3 = (C.c_float * 3)(*[float(v) for v in goal])
        _check(lib().cf_grad_host(self._h, C.c_void_p(cmds_host.data_ptr()), K, int(cmd_hold), int(n_steps), C.byref(g3),
                                  C.c_void_p(loss_host.data_ptr()), C.c_void_p(grad_host.data_ptr()), C.c_void_p(stp), st,
                                  C.c_void_p(sp), need))
        return loss_host, grad_host

    # -- sampling-based planner (cf_mppi_*) --------------------------------------------------------------------------
    def mppi_pack_best(self, mp: MppiParams, info, plan, ctrl_offset: int, row=None):
        """This shard's [score, global controller index, plan] row (device tensor of 2 + 4 H floats)."""
        if row is None:
            row = _torch().empty(2 + 4 * mp.horizon, dtype=_torch().float32, device=self.device)
        _check(lib().cf_mppi_pack_best(self._h, C.byref(mp), _dptr(info), _dptr(plan), int(ctrl_offset), _dptr(row)))
        return row

    def mppi_select(self, rows, horizon: int, out=None):
        """rows: device tensor [n_rows][2 + 4 H] -> the winning row (R31), identical whatever the row order."""
        assert rows.is_cuda and rows.is_contiguous() and rows.dtype == _torch().float32
        n_rows = rows.numel() // (2 + 4 * horizon)
        if out is None:
            out = _torch().empty(2 + 4 * horizon, dtype=_torch().float32, device=self.device)
        _check(lib().cf_mppi_select(self._h, _dptr(rows), n_rows, int(horizon), _dptr(out)))
        return out

    def mppi_params(self, horizon: int, cmd_hold: int, n_elite: int, lam: float, shift: int = 1) -> MppiParams:
        return MppiParams(C.sizeof(MppiParams), int(horizon), int(cmd_hold), int(n_elite), int(shift), float(lam))

    def _mppi_buffers(self, mp: MppiParams, want_elites: bool):
        torch = _torch()
        key = (mp.horizon, mp.n_elite)
        if getattr(self, "_mppi_key", None) != key:
            need = lib().cf_mppi_scratch_bytes(self._h, C.byref(mp))
            if need == 0:
                raise CfError(E_ARG, lib().cf_last_error().decode())
            self._mppi_scratch = torch.empty(need + 256, dtype=torch.uint8, device=self.device)
            self._mppi_need = need
            self._mppi_plan = torch.empty((mp.horizon, 4), dtype=torch.float32, device=self.device)
            self._mppi_info = torch.empty(4 * self.params.n_ctrl + 4, dtype=torch.float32, device=self.device)
            self._mppi_elites = torch.empty((self.params.n_ctrl, mp.n_elite), dtype=torch.int32, device=self.device)
            self._mppi_key = key
        sp = self._mppi_scratch.data_ptr() + (-self._mppi_scratch.data_ptr()) % 256
        return C.c_void_p(sp), self._mppi_need, (_dptr(self._mppi_elites) if want_elites else None)

    def _mppi_result(self, nominal, want_elites):
        return dict(nominal=nominal, plan=self._mppi_plan, info=self._mppi_info,
                    elites=self._mppi_elites if want_elites else None)

    def mppi_update(self, mp: MppiParams, nominal, want_elites: bool = False):
        """nominal: device tensor float32 [n_ctrl][H][4], updated IN PLACE to the warm-started sequences.  Returns
        dict(nominal, plan [H][4], info [4 n_ctrl + 4] (last word viewed as int32 = best controller), elites)."""
        sp, need, el = self._mppi_buffers(mp, want_elites)
        assert nominal.is_cuda and nominal.dtype == _torch().float32 and nominal.is_contiguous()
        assert nominal.numel() == self.params.n_ctrl * mp.horizon * 4
        _check(lib().cf_mppi_update(self._h, C.byref(mp), _dptr(nominal), _dptr(self._mppi_plan),
                                    _dptr(self._mppi_info), el, sp, need))
        return self._mppi_result(nominal, want_elites)

    def mppi_update_static(self, mp: MppiParams, nominal, plan, info, elites=None):
        """cf_mppi_update_static: the planner update for callers that may not allocate device memory (a control loop
        with a deadline, a plug-in under someone else's memory pool).  The scratch is an 8 MiB array inside libcf.so, so
        this method creates no tensor either: `plan` [H][4] float32, `info` [4 n_ctrl + 4] float32 and, optionally,
        `elites` [n_ctrl][n_elite] int32 are the caller's CUDA tensors and are written in place, `nominal`
        [n_ctrl][H][4] is updated in place.  One scratch array per GPU is shared by every simulator: keep calls that
        could overlap on the device on one stream.  CfError(CF_E_BUFFER) if the update needs more than the array holds."""
        _check(lib().cf_mppi_update_static(self._h, C.byref(mp), _dptr(nominal), _dptr(plan), _dptr(info),
                                           _dptr(elites) if elites is not None else None))

    def mppi_iterate(self, mp: MppiParams, x0, nominal, want_elites: bool = False):
        """One planning iteration: broadcast reset to x0 [D] + fused rollout + update (cf_mppi_iterate)."""
        sp, need, el = self._mppi_buffers(mp, want_elites)
        assert x0.is_cuda and x0.dtype == _torch().float32 and x0.numel() == self.D
        assert nominal.is_cuda and nominal.dtype == _torch().float32 and nominal.is_contiguous()
        assert nominal.numel() == self.params.n_ctrl * mp.horizon * 4
        _check(lib().cf_mppi_iterate(self._h, C.byref(mp), _dptr(x0), _dptr(nominal), _dptr(self._mppi_plan),
                                     _dptr(self._mppi_info), el, sp, need))
        return self._mppi_result(nominal, want_elites)

    def mppi_iterate_host(self, mp: MppiParams, x0_host, nominal, plan_host, info_host):
        """End-to-end iteration: x0_host [D], plan_host [H][4], info_host [4 n_ctrl + 4] are (pinned) CPU tensors."""
        sp, need, _ = self._mppi_buffers(mp, False)
        _check(lib().cf_mppi_iterate_host(self._h, C.byref(mp), C.c_void_p(x0_host.data_ptr()), _dptr(nominal),
                                          C.c_void_p(plan_host.data_ptr()), C.c_void_p(info_host.data_ptr()),
                                          _dptr(self._mppi_plan), _dptr(self._mppi_info), sp, need))
        return plan_host, info_host

    def nonfinite(self):
        """(number of drones with a NaN / Inf in their state, index of the first one or None) -- CF_AUX_NONFINITE."""
        w = self._aux(AUX_NONFINITE, (2,), _torch().int32).cpu().numpy().view(np.uint32)
        return int(w[0]), (None if w[1] == 0xFFFFFFFF else int(w[1]))

    def set_counters(self, counters, rec_table=None):
        """cf_set_counters: counters = the 4 words of counters(); rec_table = rec_table() (numpy / tensor) or None."""
        c = (C.c_uint32 * 4)(*[int(v) for v in counters])
        t = None
        if rec_table is not None:
            t = self._dev(np.asarray(rec_table).view(np.int32) if not isinstance(rec_table, _torch().Tensor) else rec_table,
                          _torch().int32)
            assert t.numel() == REC_TABLE_CAP
        _check(lib().cf_set_counters(self._h, C.byref(c), _dptr(t)))

    def set_copy_stream(self, stream=None):
        """cf_set_copy_stream: a torch.cuda.Stream the caller owns (kept alive here), or None for the library's own."""
        self._copy_stream = stream
        _check(lib().cf_set_copy_stream(self._h, C.c_void_p(stream.cuda_stream) if stream is not None else None))

    def rec_table(self):
        return self._aux(AUX_REC_TABLE, (REC_TABLE_CAP,), _torch().int32).cpu().numpy().view(np.uint32)

    @property
    def step_counter(self) -> int:
        return int(lib().cf_step_counter(self._h))

    def sync_counters(self):
        _check(lib().cf_sync_counters(self._h))

    def philox_dev(self, seed: int, ctr: np.ndarray):
        """ctr: uint32 [n][4] -> (words uint32 [n][4], uniforms f32 [n][4], normals f32 [n][4]) from the device code."""
        torch = _torch()
        c = torch.as_tensor(np.ascontiguousarray(ctr, dtype=np.uint32).view(np.int32), device=self.device)
        n = c.shape[0]
        words = torch.empty((n, 4), dtype=torch.int32, device=self.device)
        uni = torch.empty((n, 4), dtype=torch.float32, device=self.device)
        nrm = torch.empty((n, 4), dtype=torch.float32, device=self.device)
        _check(lib().cf_debug_philox_dev(self._h, int(seed), _dptr(c), n, _dptr(words), _dptr(uni), _dptr(nrm)))
        return words.cpu().numpy().view(np.uint32), uni.cpu().numpy(), nrm.cpu().numpy()
