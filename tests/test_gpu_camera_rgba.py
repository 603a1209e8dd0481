"""-m gpu: the camera's colour frame (mdg_render_rgba; "(N, 48, 64, 4) uint8", reading Q53) against the
float64 oracle, pixel by pixel.

A channel is floor(albedo * shade + 1/2): floating point decides an integer, the kernel in fp32 and the oracle in fp64, so the
comparison is made on the value before rounding: |gpu - albedo * shade_oracle| <= 1/2 + SHADE_TOL for every channel of every pixel
whose hit decision is not a tie (the depth test's margin).  That is bit-exact wherever the oracle's value is further than
SHADE_TOL from a rounding boundary, and lets the other pixels fall to either side.  SHADE_TOL = 0.05 of a u8 step: n.l is formed
from the unit-sphere hit point without cancellation (mdg_camera.cuh: cam_ndotl), its fp32 error is ~1e-5 for bodies a few pixels
wide and grows with distance / size; the largest deviation measured over these scenes is 0.005.  Sky and floor have no such
freedom and must match exactly; the frame must show the same primitive per pixel as the kernel's own segmentation frame.
"""
import os

import numpy as np
import pytest

import paper_2606_08039_b200 as mdg
from oracle import oracle as O
from paper_2606_08039_b200 import binding as B
from paper_2606_08039_b200 import workloads as W

pytestmark = pytest.mark.gpu
TIE = 1e-3              # the depth / segmentation tests' tie margin (tests/test_gpu_camera.py)
SHADE_TOL = 0.05
SKY, FLOOR = np.array([135, 206, 235, 255], np.uint8), np.array([138, 138, 138, 255], np.uint8)


def albedo_table(n_drones):
    k = np.arange(n_drones)
    tab = np.zeros((2 + n_drones, 3))
    tab[0], tab[1] = (135, 206, 235), (160, 160, 160)
    tab[2:] = np.stack([250 - 22 * (k % 8), 60 + 40 * ((k // 8) % 4), 40 + 26 * (k % 8)], axis=1)
    return tab


def oracle_cam_kw(c):
    return dict(H=c.height, W=c.width, fovy_deg=c.fovy_deg, offset=tuple(c.offset), znear=c.znear, zfar=c.zfar,
                body_a=c.body_radius, body_c=c.body_half_height)


def check_rgba(st32, n_envs, n_drones, rgba, seg_gpu, cam_kw, need_drone_px=1):
    want, d64, s64, mg, shade = O.render_rgba(st32.astype(np.float64), n_envs, n_drones, n_threads=os.cpu_count() or 1, **cam_kw)
    assert rgba.shape == want.shape and rgba.dtype == np.uint8
    assert (rgba[..., 3] == 255).all()
    # the frame shows what the kernel's own segmentation shows
    assert np.array_equal((rgba == SKY).all(axis=-1), seg_gpu == 0)
    assert ((rgba == FLOOR).all(axis=-1) | (seg_gpu != 1)).all()
    clear = mg >= TIE
    v = albedo_table(n_drones)[s64] * shade[..., None]
    dev = np.abs(rgba[..., :3].astype(np.float64) - v)
    assert (dev[clear] <= 0.5 + SHADE_TOL).all(), ("colour", float(dev[clear].max()), np.argwhere(clear[..., None] & (dev > 0.5 + SHADE_TOL))[:5])
    bg = clear & (s64 <= 1)
    assert np.array_equal(rgba[bg], want[bg])                       # sky and floor: exact
    drone = clear & (s64 >= 2)
    assert drone.sum() >= need_drone_px
    mism = (rgba[drone][:, :3] != want[drone][:, :3]).any(axis=1).mean() if drone.any() else 0.0
    assert mism <= 0.02, ("drone pixels on the other side of a rounding boundary", mism)
    return float(dev[clear].max() - 0.5), float(mism)


@pytest.mark.parametrize("n_envs,n_drones", [(301, 1), (64, 4), (9, 8), (5, 17), (3, 32), (40, 32)])
def test_rgba_parity_scenes(n_envs, n_drones):
    env = mdg.Env(n_envs, n_drones, W.PHYS_MJC, W.ACT_RPM, mdg.default_params(0, auto_reset=0, term_mode=W.TERM_NONE))
    env.reset(1)
    env.set_state(state=W.camera_scene(W.BASE_SEED + 70 + n_drones, n_envs, n_drones))
    cam = B.default_cam_params(env.params)
    rgba = env.render_rgba()
    _, seg = env.render_depth()
    st32 = env.get_state()["state"]
    worst, mism = check_rgba(st32, n_envs, n_drones, rgba.cpu().numpy(), seg.cpu().numpy(), oracle_cam_kw(cam), need_drone_px=0 if n_drones == 1 else 50)
    print(f"rgba {n_envs}x{n_drones}: worst deviation beyond 1/2 = {worst:.4f}, mismatching drone pixels {mism:.4f}")


@pytest.mark.parametrize("cam_over", [dict(height=30, width=52, fovy_deg=90.0, offset=(0.03, 0.01, 0.02), zfar=8.0),
                                      dict(height=64, width=128, fovy_deg=45.0, body_radius=0.12, body_half_height=0.04),
                                      dict(height=96, width=128, fovy_deg=70.0)])
def test_rgba_parity_other_intrinsics(cam_over):
    n_envs, n_drones = 21, 5
    env = mdg.Env(n_envs, n_drones, W.PHYS_MJC, W.ACT_RPM, mdg.default_params(0, auto_reset=0, term_mode=W.TERM_NONE))
    env.reset(2)
    env.set_state(state=W.camera_scene(W.BASE_SEED + 61, n_envs, n_drones, radius=0.45))
    cam = B.default_cam_params(env.params, **cam_over)
    rgba = env.render_rgba(cam)
    _, seg = env.render_depth(cam)
    check_rgba(env.get_state()["state"], n_envs, n_drones, rgba.cpu().numpy(), seg.cpu().numpy(), oracle_cam_kw(cam), need_drone_px=50)


def test_rgba_after_stepping_config_5_and_errors():
    import ctypes as C
    import torch
    wl = W.config(5).scaled(96)
    env = mdg.Env(wl.n_envs, wl.n_drones, wl.physics_mode, wl.action_type, mdg.default_params(0, **wl.params))
    env.reset(wl.seed)
    for t in range(24):
        env.step(env.gen_actions(wl.seed, t, 1.0, wl.actions[1], wl.actions[2]))
    torch.cuda.synchronize()
    rgba = env.render_rgba()
    _, seg = env.render_depth()
    check_rgba(env.get_state()["state"], wl.n_envs, wl.n_drones, rgba.cpu().numpy(), seg.cpu().numpy(),
               oracle_cam_kw(B.default_cam_params(env.params)), need_drone_px=0)
    again = env.render_rgba()
    assert torch.equal(rgba, again)                                    # deterministic
    L, h = B.lib(), env._h
    cam = B.default_cam_params(env.params)
    assert L.mdg_render_rgba(h, C.byref(cam), None) == B.MDG_EINVAL
    assert L.mdg_render_rgba(None, C.byref(cam), C.c_void_p(rgba.data_ptr())) == B.MDG_EINVAL
    assert L.mdg_render_rgba(h, C.byref(cam), C.c_void_p(rgba.data_ptr() + 4)) == B.MDG_EINVAL
    assert L.mdg_render_rgba(h, C.byref(B.default_cam_params(env.params, width=50)), C.c_void_p(rgba.data_ptr())) == B.MDG_EINVAL


def test_rgba_full_size_sampled():
    """The batch bench.py's camera leg times (16,384 envs x 4 drones = 65,536 frames, 0.8 GB), same scenes and launch
    configuration; 48 sampled envs are checked frame by frame against the oracle, the whole batch against the kernel's own
    segmentation frames."""
    import torch
    n_envs, n_drones = 16384, 4
    env = mdg.Env(n_envs, n_drones, W.PHYS_MJC, W.ACT_RPM, mdg.default_params(0, auto_reset=0, term_mode=W.TERM_NONE))
    env.reset(1)
    env.set_state(state=W.camera_scene(W.BASE_SEED + 99, n_envs, n_drones))
    rgba = env.render_rgba()
    _, seg = env.render_depth()
    torch.cuda.synchronize()
    pick = np.concatenate([[0, n_envs - 1], np.random.default_rng(0).choice(n_envs, 46, replace=False)])
    idx = torch.from_numpy(pick).cuda()
    st32 = env.get_state()["state"].reshape(n_envs, n_drones, 13)
    c = rgba.view(n_envs, n_drones, 48, 64, 4)[idx].cpu().numpy().reshape(-1, 48, 64, 4)
    s = seg.view(n_envs, n_drones, 48, 64)[idx].cpu().numpy().reshape(-1, 48, 64)
    check_rgba(st32[pick].reshape(-1, 13), len(pick), n_drones, c, s, oracle_cam_kw(B.default_cam_params(env.params)), need_drone_px=200)
    # properties that hold at any size: alpha, sky <=> background, floor colour wherever the floor is seen
    words = rgba.view(torch.int32).squeeze(-1)
    sky = int(np.array([135, 206, 235, 255], np.uint8).view(np.int32)[0])
    floor = int(np.array([138, 138, 138, 255], np.uint8).view(np.int32)[0])
    assert bool((rgba[..., 3] == 255).all())
    assert torch.equal(words == sky, seg == 0)
    assert bool(((words == floor) | (seg != 1)).all())
