"""Pins of the oracle's colour frame (oracle/camera_oracle.hpp, reading Q53; "(N, 48, 64, 4) uint8").

The frame is flat Lambert shading of the hit the depth / segmentation pins already fix, so what is pinned here is the shading:
hand values where the geometry fixes the normal (the floor, back-lit faces), a sphere's radial normals, and for tilted spheroids
the normal from finite differences of the quadric that DEFINES the body (reading Q46) - none of it goes through the oracle's
own normal formula.  scipy supplies the rotations.
"""
import math

import numpy as np
import pytest
from scipy.spatial.transform import Rotation

from oracle import oracle as O

CAM = O.CAM_DEFAULTS
L = np.array([0.36, 0.48, 0.80])            # Q53: unit vector towards the light
SKY, FLOOR = (135, 206, 235), (160, 160, 160)


def state_of(p, rpy=(0.0, 0.0, 0.0)):
    x, y, z, w = Rotation.from_euler("ZYX", [rpy[2], rpy[1], rpy[0]]).as_quat()
    return np.array([*p, w, x, y, z, 0, 0, 0, 0, 0, 0], dtype=np.float64)


def rot_of(row):
    w, x, y, z = row[3:7]
    return Rotation.from_quat([x, y, z, w]).as_matrix()


def albedo(k):
    return np.array([250 - 22 * (k % 8), 60 + 40 * ((k // 8) % 4), 40 + 26 * (k % 8)], dtype=np.float64)


def pixel_dirs(H, W, fovy_deg):
    s = 2.0 * math.tan(math.radians(fovy_deg) / 2) / H
    r, c = np.meshgrid(np.arange(H), np.arange(W), indexing="ij")
    return np.stack([np.ones((H, W)), -(c + 0.5 - W / 2) * s, -(r + 0.5 - H / 2) * s], axis=-1)


def hit_points(st, i, depth):
    Ri = rot_of(st[i])
    o = st[i, :3] + Ri @ np.array(CAM["offset"])
    return o + depth[..., None] * (pixel_dirs(48, 64, 60.0) @ Ri.T)


def boundary_distance(alb, shade):
    """Distance of the channel value closest to a u8 rounding boundary from that boundary (1/2 = as far as it gets)."""
    v = np.asarray(alb)[None, :] * np.asarray(shade).reshape(-1, 1)
    return (0.5 - np.abs(v - np.floor(v + 0.5))).min(axis=1)


def expected(alb, ndl):
    return np.floor(np.asarray(alb)[None, :] * (0.3 + 0.7 * np.maximum(0.0, ndl))[:, None] + 0.5)


def test_light_is_a_unit_vector_and_the_floor_sky_and_alpha_have_their_hand_values():
    assert abs(L @ L - 1.0) < 1e-15
    rgba, depth, seg, mg, sm = O.render_rgba(state_of((0.3, -0.2, 1.0)), 1, 1)
    assert rgba.shape == (1, 48, 64, 4) and rgba.dtype == np.uint8
    assert np.all(rgba[..., 3] == 255)
    assert np.all(rgba[0][seg[0] == 0][:, :3] == SKY)
    # floor: n = +z, n.l = 0.8, shade = 0.3 + 0.7 * 0.8 = 0.86, 160 * 0.86 = 137.6 -> 138
    assert np.all(rgba[0][seg[0] == 1][:, :3] == 138)
    assert np.allclose(sm[0][seg[0] == 1], 0.86, atol=1e-15) and np.all(sm[0][seg[0] == 0] == 1.0)


def test_depth_segmentation_and_margin_are_those_of_render_depth():
    rng = np.random.default_rng(3)
    st = np.stack([state_of(rng.uniform([-0.5, -0.5, 0.2], [0.5, 0.5, 1.2]), rng.uniform(-0.5, 0.5, 3) * [1, 1, 6]) for _ in range(5)])
    rgba, depth, seg, mg, sm = O.render_rgba(st, 1, 5)
    d0, s0, m0 = O.render_depth(st, 1, 5, with_margin=True)
    assert np.array_equal(depth, d0) and np.array_equal(seg, s0) and np.array_equal(mg, m0)


@pytest.mark.parametrize("k", [1, 9, 30])
def test_sphere_normals_are_radial(k):
    """A sphere (a = c) as drone k of the env: the normal at a hit is (hit - centre) / R, whatever the body's attitude."""
    R = 0.25
    M = k + 1
    st = np.stack([state_of((5.0 * j, 40.0, 30.0)) for j in range(M)])          # the others far away, out of sight
    st[0] = state_of((0.0, 0.0, 1.0), (0.1, -0.2, 0.7))
    ctr = np.array([0.9, 0.55, 1.2])
    st[k] = state_of(ctr, (0.4, 0.3, -1.0))
    rgba, depth, seg, mg, sm = O.render_rgba(st, 1, M, body_a=R, body_c=R)
    hit = seg[0] == 2 + k
    assert hit.sum() > 60
    n = (hit_points(st, 0, depth[0])[hit] - ctr) / R
    assert np.abs(np.linalg.norm(n, axis=1) - 1.0).max() < 1e-9
    v = albedo(k)[None, :] * (0.3 + 0.7 * np.maximum(0.0, n @ L))[:, None]
    safe = boundary_distance(albedo(k), sm[0][hit]) > 1e-6
    assert safe.mean() > 0.99
    assert np.array_equal(rgba[0][hit][safe][:, :3], np.floor(v + 0.5)[safe])
    assert (n @ L > 0.2).any() and (n @ L < 0.0).any()       # both the lit and the shadowed side are in view


def test_spheroid_normals_match_the_finite_difference_gradient_of_the_quadric():
    """Tilted oblate spheroids (a : c = 4): n = grad f / |grad f| with f(x) = |S R^T (x - p)|^2 the body's defining quadric (Q46),
    the gradient taken by central differences here."""
    a, c = 0.12, 0.03
    rng = np.random.default_rng(11)
    checked = 0
    for trial in range(5):
        M = 4
        st = np.zeros((M, 13))
        for i in range(M):
            ang = 2 * math.pi * i / M + rng.uniform(-0.2, 0.2)
            st[i] = state_of([0.6 * math.cos(ang), 0.6 * math.sin(ang), rng.uniform(0.4, 1.2)],
                             (rng.uniform(-0.6, 0.6), rng.uniform(-0.6, 0.6), ang + math.pi + rng.uniform(-0.4, 0.4)))
        rgba, depth, seg, mg, sm = O.render_rgba(st, 1, M, body_a=a, body_c=c)
        for i in range(M):
            X = hit_points(st, i, depth[i])
            for k in range(M):
                hk = seg[i] == 2 + k
                if not hk.any():
                    continue
                hk[hk] = boundary_distance(albedo(k), sm[i][hk]) > 1e-4
                Rk, pk = rot_of(st[k]), st[k, :3]
                f = lambda x: (((x - pk) @ Rk / np.array([a, a, c])) ** 2).sum(axis=-1)
                h = 1e-6
                g = np.stack([(f(X[hk] + h * e) - f(X[hk] - h * e)) / (2 * h) for e in np.eye(3)], axis=-1)
                n = g / np.linalg.norm(g, axis=1, keepdims=True)
                want = expected(albedo(k), n @ L)
                got = rgba[i][hk][:, :3].astype(np.float64)
                assert np.abs(got - want).max() <= 0            # the finite difference is good to ~1e-9: far inside the 1e-4 band left out
                checked += int(hk.sum())
    assert checked > 300


def test_back_lit_faces_get_the_ambient_term_alone():
    """A camera looking along +l sees only faces whose normals point away from the light: shade = 0.3 exactly."""
    yaw, pitch = math.atan2(L[1], L[0]), -math.asin(L[2])                        # body +x = l  (ZYX: nose up = negative pitch)
    cam = state_of((0.0, 0.0, 20.0), (0.0, pitch, yaw))
    assert np.allclose(rot_of(cam)[:, 0], L, atol=1e-12)
    k = 2
    st = np.stack([cam, state_of((50.0, 50.0, 30.0)), state_of(cam[:3] + 1.0 * L, (0.3, -0.4, 0.2))])
    rgba, depth, seg, mg, sm = O.render_rgba(st, 1, 3, body_a=0.2, body_c=0.05)
    hit = seg[0] == 2 + k
    assert hit.sum() > 40
    assert np.all(rgba[0][hit][:, :3] == np.floor(albedo(k) * 0.3 + 0.5))
    # and from the other side the same body is lit: a camera beyond it, looking back along -l
    cam2 = state_of(cam[:3] + 2.0 * L, (0.0, -pitch, yaw + math.pi))
    assert np.allclose(rot_of(cam2)[:, 0], -L, atol=1e-12)
    st2 = np.stack([cam2, st[1], st[2]])
    rgba2, depth2, seg2, _, _ = O.render_rgba(st2, 1, 3, body_a=0.2, body_c=0.05)
    hit2 = seg2[0] == 2 + k
    assert hit2.sum() > 40 and np.all(rgba2[0][hit2][:, 0].astype(int) > int(np.floor(albedo(k)[0] * 0.3 + 0.5)))


def test_albedo_palette_of_all_thirty_two_drones():
    """Each drone's colour under the ambient term alone (n.l <= 0 cannot be arranged for 31 bodies at once, so: the palette row
    of every id appears, scaled by a shade in [0.3, 1], on a wall of spheres in front of the camera)."""
    M = 32
    st = np.stack([state_of((3.0, -1.4 + 0.4 * (j % 8), 0.3 + 0.45 * (j // 8))) for j in range(M)])      # a wall of spheres, none occluded
    st[0] = state_of((0.0, 0.0, 0.9))
    rgba, depth, seg, mg, sm = O.render_rgba(st, 1, M, body_a=0.15, body_c=0.15)
    seen = 0
    for k in range(1, M):
        hk = seg[0] == 2 + k
        if hk.sum() < 3:
            continue
        seen += 1
        ratio = rgba[0][hk][:, :3].astype(np.float64) / albedo(k)[None, :]
        assert np.all(ratio >= 0.3 - 0.5 / albedo(k).min() - 1e-9) and np.all(ratio <= 1.0 + 0.5 / albedo(k).min())
        assert np.ptp(ratio, axis=1).max() <= 1.0 / albedo(k).min() + 1e-9       # the three channels share one shade
    assert seen == M - 1
