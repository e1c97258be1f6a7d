"""Pins of the depth ray-casting oracle (oracle/depth.py; reading R34): analytic distances,
hit points re-inserted into the implicit surface equations, an independent ray-marching brute force (signed-distance
sampling, no intersection formula), pixel-grid symmetry, and agreement of the two attitude conventions via scipy."""
import math

import numpy as np
import pytest
from scipy.spatial.transform import Rotation


@pytest.fixture(scope="module")
def od():
    from oracle import depth
    return depth


def ab_state(p, rpy=(0, 0, 0), n=1):
    x = np.zeros((13, n))
    x[:3] = np.asarray(p, dtype=float).reshape(3, -1)
    x[3:6] = np.asarray(rpy, dtype=float).reshape(3, -1)
    return x


def test_centre_ray_distances_to_sphere_plane_and_box(od):
    W = H = 5                                                       # odd: the centre pixel looks exactly along body +x
    sph = [[4.0, 0.0, 1.0, 0.5]]
    img = od.render(ab_state([0, 0, 1]), 1, W, H, 1.0, spheres=sph)
    assert img[0, 2, 2] == pytest.approx(3.5, rel=1e-14)
    assert img[0, 0, 0] == -1.0                                     # corner ray misses
    inside = od.render(ab_state([4.2, 0, 1]), 1, W, H, 1.0, spheres=sph)
    assert inside[0, 2, 2] == pytest.approx(0.3, rel=1e-13)         # from inside: the far surface
    theta = 0.6                                                     # positive pitch = nose down (R = Rz Ry Rx)
    img = od.render(ab_state([0, 0, 2.0], (0, theta, 0)), 1, W, H, 1.0, ground_plane=True)
    assert img[0, 2, 2] == pytest.approx(2.0 / math.sin(theta), rel=1e-13)
    img = od.render(ab_state([0, 0, 2.0], (0, -0.1, 0)), 1, W, H, 0.1, ground_plane=True)
    assert (img == -1).all()                                        # looking above the horizon
    box = [[3.0, 0.0, 1.0, 0.5, 1.0, 1.0]]
    img = od.render(ab_state([0, 0, 1]), 1, 9, 9, 0.5, boxes=box)
    dirs = od.pixel_dirs_body(9, 9, 0.5)
    np.testing.assert_allclose(img[0] * dirs[..., 0], 2.5, rtol=1e-13)      # every ray hits the front face x = 2.5
    yawed = od.render(ab_state([0, 0, 1], (0, 0, math.pi / 2)), 1, 5, 5, 0.5, boxes=[[0.0, 3.0, 1.0, 1.0, 0.5, 1.0]])
    assert yawed[0, 2, 2] == pytest.approx(2.5, rel=1e-13)          # yaw +90 deg looks along world +y


def test_pixel_grid_is_symmetric_unit_and_spans_the_field_of_view(od):
    W, H, fov = 64, 48, 1.2
    d = od.pixel_dirs_body(W, H, fov)
    np.testing.assert_allclose(np.linalg.norm(d, axis=-1), 1.0, rtol=1e-15)
    np.testing.assert_allclose(d[:, ::-1, 1], -d[..., 1], rtol=1e-15)       # left / right mirror
    np.testing.assert_allclose(d[::-1, :, 2], -d[..., 2], rtol=1e-15)       # up / down mirror
    assert d[0, 0, 1] > 0 and d[0, 0, 2] > 0                                # first pixel: up-left = body +y, +z
    # the outer EDGE of the first / last column is at half the horizontal field of view
    s = 2 * math.tan(fov / 2) / W
    assert math.atan((abs(d[H // 2, 0, 1] / d[H // 2, 0, 0])) + 0.5 * s) == pytest.approx(fov / 2, rel=1e-3)
    assert s * W / 2 == pytest.approx(math.tan(fov / 2), rel=1e-15)


def _sdf(pts, spheres, boxes, plane):
    """signed distance-like function of the scene (negative inside a primitive); plane z = 0 is a surface, not a solid"""
    v = np.full(pts.shape[:-1], np.inf)
    for s in spheres:
        v = np.minimum(v, np.linalg.norm(pts - s[:3], axis=-1) - s[3])
    for b in boxes:
        q = np.abs(pts - b[:3]) - b[3:]
        v = np.minimum(v, np.linalg.norm(np.maximum(q, 0), axis=-1) + np.minimum(q.max(-1), 0))
    return v


def test_hits_lie_on_surfaces_and_ray_marching_finds_nothing_closer(od):
    rng = np.random.default_rng(0)
    n = 6
    spheres = np.column_stack([rng.uniform(2, 6, 5), rng.uniform(-2, 2, 5), rng.uniform(0.5, 2.5, 5), rng.uniform(0.2, 0.6, 5)])
    boxes = np.column_stack([rng.uniform(2, 6, 4), rng.uniform(-2, 2, 4), rng.uniform(0.5, 2.5, 4), rng.uniform(0.1, 0.5, (4, 3))])
    st = ab_state(np.stack([rng.uniform(-0.5, 0.5, n), rng.uniform(-1, 1, n), rng.uniform(0.8, 2.0, n)]),
                  np.stack([rng.uniform(-0.3, 0.3, n), rng.uniform(-0.2, 0.5, n), rng.uniform(-0.5, 0.5, n)]), n)
    W = H = 16
    img = od.render(st, 1, W, H, 1.3, spheres=spheres, boxes=boxes, ground_plane=True, t_max=30.0)
    R = od.rotation_from_state(st, 1)
    dirs = np.einsum("nij,hwj->nhwi", R, od.pixel_dirs_body(W, H, 1.3))
    o = st[:3].T[:, None, None, :]
    hit = img > 0
    assert hit.mean() > 0.5 and (~hit).any()
    pts = o + img[..., None] * dirs
    on_solid = np.abs(_sdf(pts, spheres, boxes, False)) < 1e-9
    on_plane = np.abs(pts[..., 2]) < 1e-9
    assert (on_solid | on_plane)[hit].all()                         # every hit point is on a surface
    # brute force: sample each ray every millimetre; before the reported hit nothing is inside a solid or below the plane
    ts = np.arange(1, 12000) * 1e-3
    for idx in rng.integers(0, n * H * W, 60):
        i, v, u = np.unravel_index(idx, (n, H, W))
        ray = o[i, 0, 0] + ts[:, None] * dirs[i, v, u]
        blocked = (_sdf(ray, spheres, boxes, False) < 0) | (ray[:, 2] < 0)
        first = ts[np.argmax(blocked)] if blocked.any() else np.inf
        if img[i, v, u] > 0:
            assert first >= img[i, v, u] - 1e-9 and (first - img[i, v, u] < 2e-3 or not np.isfinite(first) or first > img[i, v, u]), (i, v, u)
            assert first - img[i, v, u] < 0.05 or not blocked.any() or abs(_sdf(pts[i, v, u][None], spheres, boxes, False)[0]) < 1e-9
        else:
            assert not blocked.any(), (i, v, u)
    # t_max cuts hits off
    near = od.render(st, 1, W, H, 1.3, spheres=spheres, boxes=boxes, ground_plane=True, t_max=3.0)
    assert ((near == -1) | (near <= 3.0)).all() and ((img > 3.0) <= (near == -1)).all()
    np.testing.assert_array_equal(near[near > 0], img[near > 0])


def test_quaternion_and_euler_states_give_the_same_image_and_the_camera_offset_moves_with_the_body(od):
    rpy = np.array([0.3, -0.2, 0.7])
    rot = Rotation.from_euler("xyz", rpy)                           # extrinsic x-y-z = Rz Ry Rx
    fp = np.zeros((17, 1)); fp[:3, 0] = [0.1, -0.2, 1.5]; fp[3:7, 0] = rot.as_quat()
    ab = ab_state([0.1, -0.2, 1.5], rpy)
    sph = [[3.0, 1.0, 1.2, 0.7], [2.0, -1.0, 2.0, 0.4]]
    a = od.render(fp, 0, 12, 10, 1.1, spheres=sph, ground_plane=True)
    b = od.render(ab, 1, 12, 10, 1.1, spheres=sph, ground_plane=True)
    np.testing.assert_allclose(a, b, rtol=1e-12)
    np.testing.assert_allclose(od.rotation_from_state(fp, 0)[0], rot.as_matrix(), atol=1e-15)
    off = np.array([0.03, 0.0, 0.01])
    c = od.render(ab, 1, 12, 10, 1.1, spheres=sph, ground_plane=True, cam_offset=off)
    moved = ab.copy(); moved[:3, 0] += rot.as_matrix() @ off
    np.testing.assert_allclose(c, od.render(moved, 1, 12, 10, 1.1, spheres=sph, ground_plane=True), rtol=1e-12)
