"""float64 ORACLE of the batched depth ray casting ("parallel rendering of depth images ... 64x64 ray
resolution across 1,024 environments"; L286-L288: ray casting and distance measurements against the scene geometry).

TEST INFRASTRUCTURE ONLY (see oracle/cfo.h).  Shares nothing with paper_2606_01478_b200/.

The paper inherits this from MJX's ray-cast pipeline and gives neither the camera model nor the test scene (MuJoCo XML,
not in the container), so the definition below is a reading (R34) and the scene is synthetic spheres, axis-aligned
boxes and an optional ground plane z = 0.  The result has a plain definition, written out here:

  camera of drone i: pinhole at  o = p_i + R_i cam_offset,  optical axis = body +x, image "right" = body -y, image
  "down" = body -z, R_i = attitude of the drone (quaternion of the first-principles state, Rz Ry Rx of the abstracted one);
  pixel (row v, column u), 0 <= v < H, 0 <= u < W, square pixels of size s = 2 tan(fov_x / 2) / W on the plane x = 1:
      d_body = normalise(1, -(u + 1/2 - W/2) s, -(v + 1/2 - H/2) s),   d = R_i d_body;
  depth[i][v][u] = the smallest t in (0, t_max] with o + t d on the surface of a primitive, or -1 if there is none
  (MuJoCo's mj_ray convention: distance along the unit ray, -1 for no hit).  A ray that starts inside a primitive hits
  its surface from the inside.

Pins: tests/test_oracle_depth.py (analytic distances to a sphere / plane / box face, hit points re-inserted into the
implicit surface equations, an independent ray-marching brute force on random scenes, symmetry of the pixel grid).
"""
from __future__ import annotations

import numpy as np


def rotation_from_state(state: np.ndarray, model: int) -> np.ndarray:
    """[D][MN] state planes -> R [MN][3][3] (body -> world)."""
    if model == 0:                                   # scalar-last unit quaternion
        x, y, z, w = state[3], state[4], state[5], state[6]
        R = np.array([[1 - 2 * (y * y + z * z), 2 * (x * y - w * z), 2 * (x * z + w * y)],
                      [2 * (x * y + w * z), 1 - 2 * (x * x + z * z), 2 * (y * z - w * x)],
                      [2 * (x * z - w * y), 2 * (y * z + w * x), 1 - 2 * (x * x + y * y)]])
    else:                                            # reading R13: R = Rz(yaw) Ry(pitch) Rx(roll)
        sr, cr, sp, cp = np.sin(state[3]), np.cos(state[3]), np.sin(state[4]), np.cos(state[4])
        sy, cy = np.sin(state[5]), np.cos(state[5])
        R = np.array([[cy * cp, cy * sp * sr - sy * cr, cy * sp * cr + sy * sr],
                      [sy * cp, sy * sp * sr + cy * cr, sy * sp * cr - cy * sr],
                      [-sp, cp * sr, cp * cr]])
    return np.moveaxis(R, 2, 0)


def pixel_dirs_body(W: int, H: int, fov_x: float) -> np.ndarray:
    """[H][W][3] unit ray directions in the body frame."""
    s = 2.0 * np.tan(0.5 * fov_x) / W
    u = np.arange(W) + 0.5 - 0.5 * W
    v = np.arange(H) + 0.5 - 0.5 * H
    d = np.stack([np.ones((H, W)), np.broadcast_to(-u * s, (H, W)), np.broadcast_to((-v * s)[:, None], (H, W))], axis=-1)
    return d / np.linalg.norm(d, axis=-1, keepdims=True)


def _ray_sphere(o, d, c, r):
    """smallest positive root of |o + t d - c|^2 = r^2 (d unit), inf if none."""
    oc = o - c
    b = (oc * d).sum(-1)
    cc = (oc * oc).sum(-1) - r * r
    disc = b * b - cc
    sq = np.sqrt(np.maximum(disc, 0.0))
    t0, t1 = -b - sq, -b + sq
    t = np.where(t0 > 0, t0, t1)
    return np.where((disc >= 0) & (t > 0), t, np.inf)


def _ray_box(o, d, c, half):
    """slab method on the axis-aligned box |x - c| <= half: entry distance, or exit distance when starting inside."""
    with np.errstate(divide="ignore", invalid="ignore"):
        inv = 1.0 / d
        ta, tb = (c - half - o) * inv, (c + half - o) * inv
    # a ray parallel to a slab (d_j = 0): inside the slab -> (-inf, +inf), outside -> never
    par = d == 0
    inside = np.abs(o - c) <= half
    lo = np.where(par, np.where(inside, -np.inf, np.inf), np.minimum(ta, tb))
    hi = np.where(par, np.where(inside, np.inf, -np.inf), np.maximum(ta, tb))
    t_in, t_out = lo.max(-1), hi.min(-1)
    t = np.where(t_in > 0, t_in, t_out)
    return np.where((t_in <= t_out) & (t > 0), t, np.inf)


def _ray_plane_z0(o, d):
    with np.errstate(divide="ignore", invalid="ignore"):
        t = -o[..., 2] / d[..., 2]
    return np.where((d[..., 2] != 0) & (t > 0), t, np.inf)


def render(state, model: int, W: int, H: int, fov_x: float, spheres=(), boxes=(), ground_plane=False,
           cam_offset=(0.0, 0.0, 0.0), t_max=np.inf) -> np.ndarray:
    """state: [D][MN] float64.  spheres: rows (cx, cy, cz, r); boxes: rows (cx, cy, cz, hx, hy, hz).  -> [MN][H][W]."""
    state = np.asarray(state, dtype=np.float64)
    R = rotation_from_state(state, model)                                         # [MN][3][3]
    p = state[:3].T                                                               # [MN][3]
    o = (p + np.einsum("nij,j->ni", R, np.asarray(cam_offset, dtype=np.float64)))[:, None, None, :]
    d = np.einsum("nij,hwj->nhwi", R, pixel_dirs_body(W, H, fov_x))               # [MN][H][W][3]
    best = np.full(d.shape[:-1], np.inf)
    for s in np.asarray(spheres, dtype=np.float64).reshape(-1, 4):
        best = np.minimum(best, _ray_sphere(o, d, s[:3], s[3]))
    for b in np.asarray(boxes, dtype=np.float64).reshape(-1, 6):
        best = np.minimum(best, _ray_box(o, d, b[:3], b[3:]))
    if ground_plane:
        best = np.minimum(best, _ray_plane_z0(o, d))
    return np.where(np.isfinite(best) & (best <= t_max), best, -1.0)
