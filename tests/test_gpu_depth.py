"""GPU parity of cf_depth (reading R34) against oracle/depth.py, pixel by pixel.

Bar: |gpu - oracle| <= 1e-4 * max(1, oracle) per pixel (float32 ray arithmetic: direction 1e-7, intersection 1e-6
relative), hit / miss must agree.  Where a ray grazes a silhouette the float32 and float64 rays may fall on different
sides of a depth discontinuity -- both answers are correct renderings -- so a pixel is exempt if the ORACLE itself
changes by more than 1 mm when the camera is rotated by +-2e-5 rad (200x the float32 direction error); such pixels must
stay below 0.5 % of the image.
"""
import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


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
def od():
    from oracle import depth
    return depth


def rotate_cameras(state, model, dyaw, dpitch):
    """the same drones with every camera turned by a small yaw / pitch (world-frame yaw, body pitch ~ small angle)"""
    from scipy.spatial.transform import Rotation
    s = state.copy()
    if model == 1:
        s[5] += dyaw; s[4] += dpitch
        return s
    q = Rotation.from_quat(s[3:7].T)
    s[3:7] = (Rotation.from_euler("z", dyaw) * q * Rotation.from_euler("y", dpitch)).as_quat().T
    return s


def check_images(od, state, model, scene, gpu_img):
    kw = dict(spheres=scene["spheres"], boxes=scene["boxes"], ground_plane=scene["ground_plane"],
              cam_offset=scene["cam_offset"], t_max=scene["t_max"] if scene["t_max"] > 0 else np.inf)
    Wd, Hd, fov = scene["width"], scene["height"], scene["fov_x"]
    ref = od.render(state, model, Wd, Hd, fov, **kw)
    g = gpu_img.astype(np.float64)
    bad = (np.abs(g - ref) > 1e-4 * np.maximum(1.0, np.abs(ref))) | ((g < 0) != (ref < 0))
    if bad.any():
        alts = [od.render(rotate_cameras(state, model, a, b), model, Wd, Hd, fov, **kw)
                for a, b in ((2e-5, 0), (-2e-5, 0), (0, 2e-5), (0, -2e-5))]
        stack = np.stack([ref] + alts)
        edge = (stack.max(0) - stack.min(0)) > 1e-3
        assert (bad <= edge).all(), f"{(bad & ~edge).sum()} interior pixels differ; first at {np.argwhere(bad & ~edge)[0]}"
    assert bad.mean() < 5e-3, bad.mean()
    assert (ref > 0).mean() > 0.3 and (ref < 0).any() or not scene["t_max"] > 0
    return bad.mean()


@pytest.mark.parametrize("model", [0, 1])
def test_depth_images_match_the_oracle(cf, W, od, model):
    wl = W.depth(seed=4, M=37, model=model, width=48, height=20)          # 960 pixels: ragged last block
    g = cf.Sim(wl.M, 1, wl.model, wl.params)
    g.reset(wl.seed)
    sc = wl.notes["scene"]
    dp = g.depth_params(**sc)
    img = g.depth(dp).cpu().numpy()
    state = g.get_state().cpu().numpy().astype(np.float64)
    frac = check_images(od, state, model, sc, img)
    # after stepping, the cameras have moved with the drones
    cmds = np.zeros((1, wl.M, 4), dtype=np.float32); cmds[..., 0] = 0.2; cmds[..., 3] = 0.3
    g.step(cmds, 40, cmd_hold=40)
    img2 = g.depth(dp).cpu().numpy()
    check_images(od, g.get_state().cpu().numpy().astype(np.float64), model, sc, img2)
    assert np.abs(img2 - img).max() > 1e-3
    print("edge-pixel fraction", frac)


def test_axis_aligned_rays_inside_starts_and_limits(cf, od):
    """level drone looking exactly along +x with an odd image: the centre column / row rays have zero components
    (the parallel-slab rule), one drone sits inside a box and one inside a sphere"""
    import torch
    g = cf.Sim(3, 1, 1, dict(integrator=0, iface=2, f_phys=500.0, f_att=500.0, init_mode=0))
    g.reset(1)
    st = np.zeros((13, 3), dtype=np.float32)
    st[:3, 0] = [0, 0, 1]; st[:3, 1] = [3.0, 0.2, 1.0]; st[:3, 2] = [6.0, -1.0, 1.5]
    st[12] = 0.26
    g.set_state(st)
    scene = dict(width=9, height=7, fov_x=1.0, spheres=[[6.0, -1.0, 1.5, 0.8]], boxes=[[3.0, 0.0, 1.0, 0.5, 1.0, 1.0]],
                 ground_plane=True, cam_offset=(0.0, 0.0, 0.0), t_max=0.0)
    img = g.depth(g.depth_params(**scene)).cpu().numpy()
    ref = od.render(st.astype(np.float64), 1, 9, 7, 1.0, spheres=scene["spheres"], boxes=scene["boxes"], ground_plane=True)
    np.testing.assert_allclose(img, ref, rtol=2e-6, atol=0)
    assert img[0, 3, 4] == pytest.approx(2.5, rel=1e-6)               # front face of the box, centre ray (d = (1, 0, 0))
    assert img[1, 3, 4] == pytest.approx(0.5, rel=1e-6)               # from inside the box: the far face
    assert img[2, 3, 4] == pytest.approx(0.8, rel=1e-6)               # from inside the sphere
    near = g.depth(g.depth_params(**dict(scene, t_max=1.0))).cpu().numpy()
    assert ((near == -1) | (near <= 1.0)).all() and (near[1] > 0).any() and near[0, 3, 4] == -1
    with pytest.raises(cf.CfError) as e:
        g.depth(g.depth_params(**dict(scene, fov_x=4.0)))
    assert e.value.code == cf.E_ARG
    # a broadcast cf_set_state is materialised before the cameras are read
    g.set_state(st[:, 1].copy(), broadcast=True)
    img_b = g.depth(g.depth_params(**scene)).cpu().numpy()
    np.testing.assert_array_equal(img_b[0], img[1]); np.testing.assert_array_equal(img_b[2], img[1])


def test_full_size_batch_sampled_against_the_oracle(cf, W, od):
    """The paper's shape: 1024 environments x 64 x 64 rays; 48 sampled environments rendered by the oracle."""
    wl = W.depth()
    g = cf.Sim(wl.M, 1, wl.model, wl.params)
    g.reset(wl.seed)
    sc = wl.notes["scene"]
    img = g.depth(g.depth_params(**sc)).cpu().numpy()
    state = g.get_state().cpu().numpy().astype(np.float64)
    assert img.shape == (1024, 64, 64) and np.isfinite(img).all()
    pick = np.concatenate([[0, 1, 1023], np.random.default_rng(0).integers(0, 1024, 45)])
    check_images(od, state[:, pick], wl.model, sc, img[pick])


def test_host_buffer_rendering_equals_device_rendering(cf, W):
    import torch
    wl = W.depth(seed=4, M=6, width=40, height=24)
    g = cf.Sim(wl.M, 1, wl.model, wl.params)
    g.reset(wl.seed)
    dp = g.depth_params(**wl.notes["scene"])
    img = g.depth(dp).cpu().numpy()
    out = torch.empty((wl.M, 24, 40), dtype=torch.float32, pin_memory=True)
    g.depth_host(dp, out)                                             # the simulator's current poses
    assert np.array_equal(out.numpy(), img)
    st = g.get_state().cpu()
    st[0] += 0.25                                                     # poses supplied by the host: every camera moved in x
    g.depth_host(dp, out, state_host=st.pin_memory())
    g2 = cf.Sim(wl.M, 1, wl.model, wl.params)
    g2.reset(wl.seed)
    g2.set_state(st.numpy())
    assert np.array_equal(out.numpy(), g2.depth(dp).cpu().numpy()) and not np.array_equal(out.numpy(), img)
