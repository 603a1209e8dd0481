"""-m gpu: the onboard depth / segmentation camera (mdg_render_depth) against the float64 ray-casting oracle.

Both sides render the SAME fp32 state (the GPU's planes read back and widened).  Segmentation ids are integers decided by
floating-point comparisons, so they are compared bit-exactly except on pixels the oracle itself marks as ties (its margin:
the relative distance of the closest decision - silhouette, near / far clip, depth order, floor side - to its threshold);
those are counted and bounded.  Depth on every pixel that is not a tie: spheroid hits |dt| <= 1e-4 t (fp32 ray
setup and the closest-approach form of the quadratic keep the error near 1e-5 t); floor hits |dt| <= (1e-5 + 1e-6 t / o_z) t,
because t = o_z / |d_z| and the fp32 world-z component d_z of the ray (a three-term sum of O(1) products of rotation-matrix
entries that are themselves rounded) carries an absolute error of a few 1e-7: a ray that grazes the floor far away from a low
camera is that ill-conditioned in any fp32 implementation (equivalently: the image is the oracle's for ray directions moved
by less than 1e-6 rad).
"""
import ctypes as C

import numpy as np
import pytest

import paper_2606_08039_b200 as mdg
from oracle import oracle as O
from paper_2606_08039_b200 import binding as B
from paper_2606_08039_b200 import workloads as W

pytestmark = pytest.mark.gpu
TIE, RTOL = 1e-3, 1e-4


def make_env(n_envs, n_drones, model=0):
    return mdg.Env(n_envs, n_drones, W.PHYS_MJC, W.ACT_RPM, mdg.default_params(model, auto_reset=0, term_mode=W.TERM_NONE))


def check_against_oracle(st32, n_envs, n_drones, depth, seg, cam_kw, max_tie_frac=0.005, need_ids=()):
    import os
    d64, s64, mg = O.render_depth(st32.astype(np.float64), n_envs, n_drones, n_threads=os.cpu_count() or 1, with_margin=True, **cam_kw)
    clear = mg >= TIE
    assert 1.0 - clear.mean() <= max_tie_frac, ("tie fraction", 1.0 - clear.mean())
    bad = (seg != s64) & clear
    assert not bad.any(), ("segmentation", int(bad.sum()), np.argwhere(bad)[:5], seg[bad][:5], s64[bad][:5], mg[bad][:5])
    same = clear & (seg == s64)
    err = np.abs(depth.astype(np.float64) - d64) / d64
    st = st32.astype(np.float64)
    w, x, y, z = st[:, 3], st[:, 4], st[:, 5], st[:, 6]
    off = cam_kw.get("offset", O.CAM_DEFAULTS["offset"])
    o_z = st[:, 2] + 2 * (x * z - w * y) * off[0] + 2 * (y * z + w * x) * off[1] + (1 - 2 * (x * x + y * y)) * off[2]
    tol = np.where(s64 == 1, 1e-5 + 1e-6 * d64 / np.maximum(o_z, 1e-9)[:, None, None], RTOL)
    assert (err <= tol)[same].all(), ("depth", float((err / tol)[same].max()), np.argwhere(same & (err > tol))[:5])
    # ties: the id must still be one a neighbouring decision could give (a real primitive or background) and the depth in range
    assert seg.max() <= 1 + n_drones and depth.min() >= cam_kw.get("znear", O.CAM_DEFAULTS["znear"]) * (1 - 1e-6)
    for i in need_ids:
        assert (s64 == i).any(), f"scene never shows id {i}"
    return float((err / tol)[same].max()), float(1.0 - clear.mean())


def oracle_cam_kw(c):
    return dict(H=c.height, W=c.width, fovy_deg=c.fovy_deg, offset=tuple(c.offset), znear=c.znear, zfar=c.zfar,
                body_a=c.body_radius, body_c=c.body_half_height)


@pytest.mark.parametrize("n_envs,n_drones", [(37, 3), (64, 4), (9, 8), (301, 1), (3, 32), (5, 17)])
def test_camera_parity_scenes(n_envs, n_drones):
    env = make_env(n_envs, n_drones)
    env.reset(1)
    env.set_state(state=W.camera_scene(W.BASE_SEED + 40 + n_drones, n_envs, n_drones))
    depth, seg = env.render_depth()
    st32 = env.get_state()["state"]
    cam = B.default_cam_params(env.params)
    ids = (0, 1) if n_drones == 1 else (0, 1, 2, 1 + n_drones)
    check_against_oracle(st32, n_envs, n_drones, depth.cpu().numpy(), seg.cpu().numpy(), oracle_cam_kw(cam), need_ids=ids)


def test_camera_defaults_follow_the_paper():
    c = B.default_cam_params()
    assert (c.height, c.width, c.fovy_deg) == (48, 64, 60.0) and tuple(c.offset) == (np.float32(0.02), 0.0, 0.0)
    assert abs(c.body_radius - (0.0397 + 0.02325)) < 1e-7                                                          # Table 2
    r = B.default_cam_params(mdg.default_params(W.MODEL_RACE))
    assert abs(r.body_radius - (0.125 + 0.0635)) < 1e-6


@pytest.mark.parametrize("cam_over", [dict(height=30, width=52, fovy_deg=90.0, offset=(0.03, 0.01, 0.02), zfar=8.0),
                                      dict(height=7, width=4, fovy_deg=20.0, znear=0.3),
                                      dict(height=96, width=128, body_radius=0.05, body_half_height=0.11)])
def test_camera_parity_other_intrinsics(cam_over):
    n_envs, n_drones = 21, 5
    env = make_env(n_envs, n_drones)
    env.reset(2)
    env.set_state(state=W.camera_scene(W.BASE_SEED + 60, n_envs, n_drones, radius=0.45))
    cam = B.default_cam_params(env.params, **cam_over)
    depth, seg = env.render_depth(cam)
    check_against_oracle(env.get_state()["state"], n_envs, n_drones, depth.cpu().numpy(), seg.cpu().numpy(), oracle_cam_kw(cam),
                         max_tie_frac=0.02)


@pytest.mark.parametrize("c", [4, 5])
def test_camera_after_stepping_a_benchmark_config(c):
    """The call reads the planes the step kernel writes: render after chained steps of configs 4 (8 drones on a grid, all facing
    +x) and 5 (formation circle), on the same stream, without a host synchronisation in between."""
    import torch
    wl = W.config(c).scaled(96)
    env = mdg.Env(wl.n_envs, wl.n_drones, wl.physics_mode, wl.action_type, mdg.default_params(0, **wl.params))
    env.reset(wl.seed)
    base = W.hover_rpm_f32() if wl.actions[0] == "hover_scale" else 1.0
    for t in range(10):
        env.step(env.gen_actions(wl.seed, t, base, wl.actions[1], wl.actions[2]))
    depth, seg = env.render_depth()
    env.step(env.gen_actions(wl.seed, 10, base, wl.actions[1], wl.actions[2]))      # a later step must not disturb the images
    d2, s2 = env.render_depth()
    torch.cuda.synchronize()
    assert not torch.equal(depth, d2)
    # replay the first 10 steps on a second handle to read the state the first render saw
    ref = mdg.Env(wl.n_envs, wl.n_drones, wl.physics_mode, wl.action_type, mdg.default_params(0, **wl.params))
    ref.reset(wl.seed)
    for t in range(10):
        ref.step(ref.gen_actions(wl.seed, t, base, wl.actions[1], wl.actions[2]))
    st32 = ref.get_state()["state"]
    check_against_oracle(st32, wl.n_envs, wl.n_drones, depth.cpu().numpy(), seg.cpu().numpy(), oracle_cam_kw(B.default_cam_params(env.params)),
                         need_ids=(0, 1, 3))


def test_camera_depth_only_seg_only_and_errors():
    import torch
    env = make_env(16, 4)
    env.reset(3)
    env.set_state(state=W.camera_scene(5, 16, 4))
    depth, seg = env.render_depth()
    d_only, none = env.render_depth(want_seg=False)
    none2, s_only = env.render_depth(want_depth=False)
    assert none is None and none2 is None and torch.equal(d_only, depth) and torch.equal(s_only, seg)
    L, h = B.lib(), env._h
    cam = B.default_cam_params(env.params)
    dp, sp = C.c_void_p(depth.data_ptr()), C.c_void_p(seg.data_ptr())
    assert L.mdg_render_depth(h, C.byref(cam), None, None) == B.MDG_EINVAL
    assert L.mdg_render_depth(None, C.byref(cam), dp, sp) == B.MDG_EINVAL
    assert L.mdg_render_depth(h, C.byref(cam), C.c_void_p(depth.data_ptr() + 4), sp) == B.MDG_EINVAL
    assert L.mdg_render_depth(h, C.byref(cam), dp, C.c_void_p(seg.data_ptr() + 1)) == B.MDG_EINVAL
    for bad in (dict(width=50), dict(height=0), dict(fovy_deg=180.0), dict(znear=0.0), dict(zfar=0.005), dict(body_radius=0.0), dict(struct_size=8)):
        assert L.mdg_render_depth(h, C.byref(B.default_cam_params(env.params, **bad)), dp, sp) == B.MDG_EINVAL, bad
    assert b"mdg_render_depth" in L.mdg_last_error()
    n0 = env.launch_count
    env.render_depth(depth=depth, seg=seg)
    assert env.launch_count == n0 + 1


def test_camera_full_size_sampled():
    """BASELINE.json's largest batch (65,536 envs x 4 drones = 262,144 cameras, 4 GB of depth + 0.8 GB of segmentation), in the
    launch configuration bench.py times; 48 sampled envs are checked image by image against the oracle."""
    import torch
    n_envs, n_drones = 65536, 4
    env = make_env(n_envs, n_drones)
    env.reset(4)
    st = W.camera_scene(W.BASE_SEED + 99, n_envs, n_drones)
    env.set_state(state=st)
    depth, seg = env.render_depth()
    torch.cuda.synchronize()
    rng = np.random.default_rng(0)
    pick = np.concatenate([[0, n_envs - 1], rng.choice(n_envs, 46, replace=False)])
    st32 = env.get_state()["state"].reshape(n_envs, n_drones, 13)
    d = depth.view(n_envs, n_drones, 48, 64)[torch.from_numpy(pick).cuda()].cpu().numpy().reshape(-1, 48, 64)
    s = seg.view(n_envs, n_drones, 48, 64)[torch.from_numpy(pick).cuda()].cpu().numpy().reshape(-1, 48, 64)
    check_against_oracle(st32[pick].reshape(-1, 13), len(pick), n_drones, d, s, oracle_cam_kw(B.default_cam_params(env.params)))
    # properties that hold at any size: ids in range, depth within [znear, zfar], background <=> zfar
    assert int(seg.max()) <= 1 + n_drones and float(depth.min()) >= 0.01 and float(depth.max()) == 50.0
    assert torch.equal(seg == 0, depth == 50.0)
