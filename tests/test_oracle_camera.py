"""Pins of the camera oracle (oracle/camera_oracle.hpp, readings Q45-Q48).

The ray caster is a definition written out, so it is pinned to what the geometry fixes independently of it: forward
pinhole projection (tests/golden/camera_bearings.txt), similar triangles for the floor, the angular size of a sphere,
points reconstructed from depth lying on their primitive, symmetries, and a brute-force march along each ray that uses
only the implicit inside test.  scipy's Rotation supplies rotations here so that no helper of the oracle is re-used.
"""
import math
import os

import numpy as np
import pytest
from scipy.spatial.transform import Rotation

from oracle import oracle as O

GOLD = os.path.join(os.path.dirname(__file__), "golden", "camera_bearings.txt")
CAM = O.CAM_DEFAULTS
S48 = 2.0 * math.tan(math.radians(30.0)) / 48.0


def state_of(p, rpy=(0.0, 0.0, 0.0)):
    """One drone row [p, q(w x y z), v, w] with the ZYX attitude rpy."""
    x, y, z, w = Rotation.from_euler("ZYX", [rpy[2], rpy[1], rpy[0]]).as_quat()
    return np.array([*p, w, x, y, z, 0, 0, 0, 0, 0, 0], dtype=np.float64)


def gold():
    bearings, floor = [], []
    for line in open(GOLD):
        t = line.split()
        if not t or t[0].startswith("#"):
            continue
        if t[0] == "floor":
            floor.append((int(t[1]), float(t[2])))
        else:
            bearings.append(tuple(float(x) for x in t))
    return bearings, floor


def test_floor_rows_level_camera():
    # camera origin = p + (0.02, 0, 0): 1 m above the floor, level
    depth, seg = O.render_depth(state_of((0.3, -0.2, 1.0)), 1, 1)
    assert depth.shape == (1, 48, 64) and seg.dtype == np.uint8
    assert np.all(seg[0, :25] == 0) and np.all(depth[0, :25] == CAM["zfar"])     # horizon: rows above it and row 24 (83 m > zfar)
    assert np.all(seg[0, 25:] == 1)
    for r, d in gold()[1]:
        assert np.allclose(depth[0, r, :], d, rtol=2e-7), r                     # the same along the whole row: depth is axial, not radial


@pytest.mark.parametrize("yaw", [0.0, 1.1])
def test_forward_projection_bearings(yaw):
    cam = state_of((0.0, 0.0, 30.0), (0.0, 0.0, yaw))
    o = np.array([0.02 * math.cos(yaw), 0.02 * math.sin(yaw), 30.0])
    for az, el, row, col in gold()[0]:
        a, e = math.radians(az) + yaw, math.radians(el)
        tgt = o + 1.0 * np.array([math.cos(e) * math.cos(a), math.cos(e) * math.sin(a), math.sin(e)])
        depth, seg = O.render_depth(np.stack([cam, state_of(tgt)]), 1, 2, body_a=0.02, body_c=0.02)
        rr, cc = np.nonzero(seg[0] == 3)
        assert len(rr) > 0, (az, el)
        assert (int(row), int(col)) in set(zip(rr.tolist(), cc.tolist())), (az, el, rr, cc)
        assert np.all(np.hypot(rr + 0.5 - row, cc + 0.5 - col) < 1.6), (az, el, rr, cc)
        assert np.all(seg[0][seg[0] != 3] == 0)


def test_on_axis_sphere_size_and_depth():
    R, d = 0.3, 1.0
    cam = state_of((-0.02, 0.0, 40.0))
    depth, seg = O.render_depth(np.stack([cam, state_of((d, 0.0, 40.0))]), 1, 2, body_a=R, body_c=R)
    hit = seg[0] == 3
    r_px = math.tan(math.asin(R / d)) / S48                 # the silhouette of an on-axis sphere is a circle of this radius
    assert abs(hit.sum() - math.pi * r_px ** 2) <= 0.3 * 2 * math.pi * r_px
    rr, cc = np.nonzero(hit)
    assert abs(rr.mean() + 0.5 - 24) < 1e-9 and abs(cc.mean() + 0.5 - 32) < 1e-9
    assert d - R <= depth[0][hit].min() < d - R + 2e-3
    assert depth[0][hit].max() < d                           # front face only
    assert np.all(depth[0][~hit] == CAM["zfar"])


def random_scene(rng, M):
    st = np.zeros((M, 13))
    for i in range(M):
        st[i] = state_of(rng.uniform([-0.6, -0.6, 0.3], [0.6, 0.6, 1.5]), rng.uniform(-0.6, 0.6, 3) * [1, 1, 5])
    return st


def ring_scene(rng, M, radius=0.6):
    """Drones on a circle, each looking roughly at the centre, so that every camera sees some of the others."""
    st = np.zeros((M, 13))
    for i in range(M):
        a = 2 * math.pi * i / M + rng.uniform(-0.2, 0.2)
        p = [radius * math.cos(a), radius * math.sin(a), rng.uniform(0.4, 1.2)]
        st[i] = state_of(p, (rng.uniform(-0.3, 0.3), rng.uniform(-0.3, 0.3), a + math.pi + rng.uniform(-0.4, 0.4)))
    return st


def pixel_dirs(H, W, fovy_deg):
    s = 2.0 * math.tan(math.radians(fovy_deg) / 2) / H
    r, c = np.meshgrid(np.arange(H), np.arange(W), indexing="ij")
    return np.stack([np.ones((H, W)), -(c + 0.5 - W / 2) * s, -(r + 0.5 - H / 2) * s], axis=-1)


def rot_of(row):
    w, x, y, z = row[3:7]
    return Rotation.from_quat([x, y, z, w]).as_matrix()


def test_reconstructed_points_lie_on_their_primitive():
    rng = np.random.default_rng(7)
    a, c = 0.12, 0.03
    seen = set()
    for _ in range(6):
        M = 4
        st = ring_scene(rng, M) if _ % 2 else random_scene(rng, M)
        depth, seg = O.render_depth(st, 1, M, body_a=a, body_c=c)
        for i in range(M):
            Ri = rot_of(st[i])
            o = st[i, :3] + Ri @ np.array(CAM["offset"])
            X = o + depth[i][..., None] * (pixel_dirs(48, 64, 60.0) @ Ri.T)
            fl = seg[i] == 1
            assert np.abs(X[fl][:, 2]).max(initial=0) < 1e-9
            for k in range(M):
                hk = seg[i] == 2 + k
                assert not (k == i and hk.any())
                if hk.any():
                    seen.add(k)
                    y = (X[hk] - st[k, :3]) @ rot_of(st[k]) / np.array([a, a, c])
                    assert np.abs((y ** 2).sum(axis=1) - 1.0).max() < 1e-8
    assert len(seen) == 4


def test_brute_force_march_small_image():
    rng = np.random.default_rng(11)
    a, c, H, W = 0.15, 0.05, 6, 8
    st = random_scene(rng, 3)
    st[:, :3] = [[0, 0, 0.6], [0.8, 0.1, 0.65], [0.9, -0.3, 0.5]]
    st[0] = state_of((0, 0, 0.6), (0.05, 0.1, 0.0))
    depth, seg = O.render_depth(st, 1, 3, H=H, W=W, body_a=a, body_c=c, zfar=6.0)
    ts = np.arange(CAM["znear"], 6.0, 5e-4)
    Ri = rot_of(st[0])
    o = st[0, :3] + Ri @ np.array(CAM["offset"])
    dirs = pixel_dirs(H, W, 60.0) @ Ri.T
    assert (seg[0] >= 2).any() and (seg[0] == 1).any()
    for r in range(H):
        for col in range(W):
            X = o + ts[:, None] * dirs[r, col]
            inside = np.zeros((len(ts), 3), bool)
            inside[:, 0] = X[:, 2] <= 0.0
            for k in (1, 2):
                y = (X - st[k, :3]) @ rot_of(st[k]) / np.array([a, a, c])
                inside[:, k] = (y ** 2).sum(axis=1) <= 1.0
            first = inside.any(axis=1).argmax() if inside.any() else -1
            if first < 0:
                assert seg[0, r, col] == 0 and depth[0, r, col] == 6.0
            elif seg[0, r, col] != 0:
                assert abs(ts[first] - depth[0, r, col]) < 1e-3, (r, col)
                assert inside[first, 0 if seg[0, r, col] == 1 else seg[0, r, col] - 2]
            else:                                                  # a grazing ray may be caught by the march only
                assert inside[first:first + 40].sum() < 40


def test_yaw_corotation_invariance():
    rng = np.random.default_rng(3)
    st = ring_scene(rng, 4)
    d0, s0 = O.render_depth(st, 1, 4, body_a=0.12, body_c=0.03)
    psi = 0.83
    Rz = Rotation.from_euler("z", psi)
    st2 = st.copy()
    st2[:, :3] = Rz.apply(st[:, :3])
    for i in range(4):
        w, x, y, z = st[i, 3:7]
        x2, y2, z2, w2 = (Rz * Rotation.from_quat([x, y, z, w])).as_quat()
        st2[i, 3:7] = [w2, x2, y2, z2]
    d1, s1 = O.render_depth(st2, 1, 4, body_a=0.12, body_c=0.03)
    assert np.array_equal(s0, s1) and np.allclose(d0, d1, rtol=1e-9)
    assert len(np.unique(s0)) >= 3


def test_roll_by_pi_flips_the_image():
    rng = np.random.default_rng(5)
    st = random_scene(rng, 3)
    st[0] = state_of((0.0, 0.0, 0.8), (0.0, 0.2, 0.3))
    d0, s0 = O.render_depth(st, 1, 3, body_a=0.12, body_c=0.03)
    st[0] = state_of((0.0, 0.0, 0.8), (math.pi, -0.2, 0.3 + math.pi))   # same optical axis, rolled by pi about it ...
    # ... built differently to make sure: q' = q * rot_x(pi)
    w, x, y, z = state_of((0, 0, 0), (0.0, 0.2, 0.3))[3:7]
    x2, y2, z2, w2 = (Rotation.from_quat([x, y, z, w]) * Rotation.from_euler("x", math.pi)).as_quat()
    st[0, 3:7] = [w2, x2, y2, z2]
    d1, s1 = O.render_depth(st, 1, 3, body_a=0.12, body_c=0.03)
    assert np.array_equal(s1[0], s0[0, ::-1, ::-1]) and np.allclose(d1[0], d0[0, ::-1, ::-1], rtol=1e-9)
    assert (s0[0] == 1).any()


def test_occlusion_order_and_near_clip():
    cam = state_of((-0.02, 0.0, 40.0))
    near, far = state_of((1.0, 0.0, 40.0)), state_of((2.0, 0.0, 40.0))
    d, s = O.render_depth(np.stack([cam, near, far]), 1, 3, body_a=0.1, body_c=0.1)
    assert s[0, 24, 32] == 3 and abs(d[0, 24, 32] - 0.9) < 2e-3
    assert not (s[0] == 4).any()                                      # the far sphere is angularly smaller: fully hidden
    d2, s2 = O.render_depth(np.stack([cam, far, near]), 1, 3, body_a=0.1, body_c=0.1)
    assert s2[0, 24, 32] == 4 and np.array_equal(d[0], d2[0])         # order in the list does not matter, ids follow the drones
    assert (s[1] == 4).any() and not (s[1] == 2).any()                # the middle drone looks along +x: sees the far one, not the camera drone
    assert np.all(s[2] == 0)                                          # the far one sees nothing
    # near clip: a sphere whose front face is closer than znear is not drawn (front faces only, reading Q46)
    d4, s4 = O.render_depth(np.stack([cam, state_of((0.05, 0.0, 40.0))]), 1, 2, body_a=0.06, body_c=0.06)
    assert np.all(s4[0] == 0) and np.all(d4[0] == CAM["zfar"])


def test_ring_of_far_sphere_around_near_sphere():
    cam = state_of((-0.02, 0.0, 40.0))
    near, far = state_of((1.0, 0.0, 40.0)), state_of((2.0, 0.0, 40.0))
    # per-drone sizes are shared, so make the far one angularly larger by an oblate body seen along its axis:
    # both pitched by 90 deg show discs of radius a; the near one is moved off-axis instead
    near = state_of((1.0, 0.12, 40.0))
    d, s = O.render_depth(np.stack([cam, near, far]), 1, 3, body_a=0.1, body_c=0.1)
    both = (s[0] == 3) | (s[0] == 4)
    assert (s[0] == 3).any() and (s[0] == 4).any()
    # inside the overlap of the two discs the near id wins: every pixel within both angular radii carries id 3
    dirs = pixel_dirs(48, 64, 60.0)
    u = dirs / np.linalg.norm(dirs, axis=-1, keepdims=True)
    def within(centre, R):
        v = np.array(centre) - np.array([0.0, 0.0, 40.0])
        return np.arccos(np.clip(u @ (v / np.linalg.norm(v)), -1, 1)) < math.asin(R / np.linalg.norm(v))
    in_near, in_far = within((1.0, 0.12, 40.0), 0.1), within((2.0, 0.0, 40.0), 0.1)
    assert (in_near & in_far).any()
    assert np.all(s[0][in_near] == 3) and np.all(s[0][in_far & ~in_near] == 4) and np.all(s[0][~in_near & ~in_far] == 0)
    assert np.array_equal(both, in_near | in_far)


def test_spheroid_aspect_edge_on_and_along_axis():
    cam = state_of((-0.02, 0.0, 40.0))
    a, c, d, H, W = 0.3, 0.06, 2.0, 240, 320
    s = 2.0 * math.tan(math.radians(30.0)) / H
    dep, seg = O.render_depth(np.stack([cam, state_of((d, 0.0, 40.0))]), 1, 2, body_a=a, body_c=c, H=H, W=W)
    hit = seg[0] == 3
    cols, rows = hit.any(axis=0).sum(), hit.any(axis=1).sum()
    assert abs(cols - 2 * math.tan(math.asin(a / d)) / s) <= 2          # edge-on: width from the equatorial circle of radius a
    assert abs(rows - 2 * (c / math.sqrt(d * d - a * a * 0)) / s) <= 2   # height ~ 2c/d (c << d)
    assert abs(hit.sum() - math.pi * (cols / 2) * (rows / 2)) < 0.08 * hit.sum()    # an ellipse
    # pitched by 90 deg its axis points at the camera: a disc of radius a at distance d, front face at d - c
    dep2, seg2 = O.render_depth(np.stack([cam, state_of((d, 0.0, 40.0), (0.0, math.pi / 2, 0.0))]), 1, 2, body_a=a, body_c=c, H=H, W=W)
    hit2 = seg2[0] == 3
    cols2, rows2 = hit2.any(axis=0).sum(), hit2.any(axis=1).sum()
    assert abs(cols2 - rows2) <= 1 and abs(cols2 - 2 * (a / d) / s) <= 3
    assert d - c <= dep2[0][hit2].min() < d - c + 1e-3


def test_single_drone_and_camera_below_floor():
    d, s = O.render_depth(state_of((0.0, 0.0, 0.5), (0.0, 0.4, 0.0)), 1, 1)          # pitched nose-down: more floor
    d0, s0 = O.render_depth(state_of((0.0, 0.0, 0.5)), 1, 1)
    assert set(np.unique(s)) <= {0, 1} and (s == 1).sum() > (s0 == 1).sum()
    d1, s1 = O.render_depth(state_of((0.0, 0.0, 0.0), (0.0, 0.4, 0.0)), 1, 1)        # on the floor, camera origin below z = 0
    assert np.all(s1 == 0) and np.all(d1 == CAM["zfar"])


def test_margin_flags_only_a_thin_band():
    rng = np.random.default_rng(2)
    st = np.concatenate([ring_scene(rng, 4) for _ in range(8)])
    d, s, m = O.render_depth(st, 8, 4, with_margin=True)
    assert (m < 1e-3).mean() < 0.01 and (s >= 2).mean() > 0.002
    d2, s2 = O.render_depth(st, 8, 4, n_threads=3)
    assert np.array_equal(d, d2) and np.array_equal(s, s2)
