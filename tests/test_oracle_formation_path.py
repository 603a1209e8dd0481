"""Pins of the oracle's moving formation centre ("the formation centre tracks a closed polygonal path"; reading
Q52: constant speed along the closed polygon from vertex 0 at episode time 0).  Expected positions are worked out by hand for a
unit square and a 3-4-5 triangle; rewards and terminations are those of formation states built by hand around them."""
import math

import numpy as np

from oracle_util import make_env
from paper_2606_08039_b200 import workloads as W

HOVER = W.hover_rpm_f32()
BASE = dict(reward_mode=W.REW_FORMATION, term_mode=W.TERM_FORMATION, target_mode=W.TGT_CIRCLE, form_radius=0.3,
            reset_layout=W.LAYOUT_CIRCLE, circle_radius=0.3, reset_half=[0, 0, 0], term_dist=3.0, episode_len_s=100.0, auto_reset=0)
SQUARE = [0, 0, 1, 1, 0, 1, 1, 1, 1, 0, 1, 1] + [0] * 12            # unit square at z = 1, perimeter 4
TRI = [0, 0, 1, 3, 0, 1, 3, 4, 2] + [0] * 15                          # sides 3, sqrt(16 + 1), sqrt(9 + 16 + 1)


def centre_of(env, M):
    t = env.targets.reshape(-1, M, 4)[0]
    return t[:, :3].mean(axis=0), t                                   # the slots are symmetric about the centre (M even or odd)


def test_centre_walks_the_closed_square_at_constant_speed():
    M = 4
    env, _ = make_env(n_drones=M, form_path_n=4, form_path=SQUARE, form_speed=0.5, reset_center=[0, 0, 1], **BASE)
    c, t = centre_of(env, M)
    assert np.allclose(c, [0, 0, 1], atol=1e-12)
    assert np.allclose(t[:, :3], [[0.3, 0, 1], [0, 0.3, 1], [-0.3, 0, 1], [0, -0.3, 1]], atol=1e-12)   # slots of PAPER.md:325 about vertex 0
    a = np.full((M, 4), HOVER, dtype=np.float32)
    # hand table: speed 0.5 m/s, sides of 1 m -> a vertex every 2 s, the lap closes after 8 s
    want = {1.0: [0.5, 0, 1], 2.0: [1, 0, 1], 3.0: [1, 0.5, 1], 4.0: [1, 1, 1], 5.5: [0.25, 1, 1], 6.0: [0, 1, 1], 7.0: [0, 0.5, 1],
            8.0: [0, 0, 1], 9.0: [0.5, 0, 1], 0.5: [0.25, 0, 1]}
    for k in range(1, 9 * 48 + 1):
        env.step(a)
        tau = k / 48.0
        if tau in want:
            c, t = centre_of(env, M)
            assert np.allclose(c, want[tau], atol=1e-9), (tau, c)
            assert np.allclose(t[1, :3] - c, [0, 0.3, 0], atol=1e-9)


def test_unequal_sides_and_a_climbing_leg():
    M = 3
    env, _ = make_env(n_drones=M, form_path_n=3, form_path=TRI, form_speed=1.0, reset_center=[0, 0, 1], **BASE)
    a = np.full((M, 4), HOVER, dtype=np.float32)
    l2, l3 = math.sqrt(17.0), math.sqrt(26.0)
    checks = {48 * 3: [3, 0, 1],                                        # end of the first side after 3 s
              48 * 5: [3, 4 * 2 / l2, 1 + 2 / l2],                      # 2 m up the second side
              48 * 12: None}
    for k in range(1, 48 * 12 + 1):
        env.step(a)
        if k in checks and checks[k] is not None:
            assert np.allclose(centre_of(env, M)[0], checks[k], atol=1e-9), k
    s = 12.0 - 3.0 - l2                                                 # arc length into the third side after 12 s (perimeter 12.22)
    assert 0 < s < l3
    assert np.allclose(centre_of(env, M)[0], np.array([3, 4, 2]) + s / l3 * (np.array([0, 0, 1]) - np.array([3, 4, 2])), atol=1e-9)


def test_reward_and_termination_ride_on_the_moving_centre():
    M = 4
    env, _ = make_env(n_drones=M, form_path_n=4, form_path=SQUARE, form_speed=0.5, reset_center=[0, 0, 1], **BASE)
    a = np.full((M, 4), HOVER, dtype=np.float32)
    for _ in range(95):
        env.step(a)
    # next step ends at tau = 2 s: centre (1, 0, 1).  Park the drones 0.02 m above the slots they will be asked to hold.
    slots = np.array([[1.3, 0, 1], [1, 0.3, 1], [0.7, 0, 1], [1, -0.3, 1]])
    s = env.state
    s[:, 0:3] = slots + [0, 0, 0.02]; s[:, 3:7] = [1, 0, 0, 0]; s[:, 7:13] = 0
    env.state = s
    env.step(a)
    obs, rew, done, _ = env.outputs()
    z = env.state[:, 2]
    assert np.abs(z - 1.02).max() < 1e-6                                # hover thrust: parked
    assert abs(rew[0] + np.abs(z - 1.0).sum()) < 1e-9 and done[0] == 0  # -sum |p_i - slot_i|, pair distances exact
    # the static reading (Q26) would have scored the same state from (0, 0, 1): about -4 m
    env2, _ = make_env(n_drones=M, reset_center=[0, 0, 1], form_center=[0, 0, 1], **BASE)
    s2 = env2.state; s2[:] = s; env2.state = s2
    env2.step(a)
    assert env2.outputs()[1][0] < -3.5
    # termination: 2.9 m from the moving centre is inside, 3.1 m is out - although the static centre says the opposite
    for off, want in ((2.9, 0), (3.1, 1)):
        env3, _ = make_env(n_drones=M, form_path_n=4, form_path=SQUARE, form_speed=0.5, reset_center=[0, 0, 1], term_center=[0, 0, 1], **BASE)
        for _ in range(95):
            env3.step(a)
        s3 = env3.state
        s3[:, 0:3] = slots; s3[:, 3:7] = [1, 0, 0, 0]; s3[:, 7:13] = 0
        s3[0, 0:3] = [1 + off, 0, 1]
        env3.state = s3
        env3.step(a)
        assert env3.outputs()[2][0] == want, off


def test_static_centre_is_the_default_and_a_reset_returns_to_vertex_zero():
    M = 4
    env, _ = make_env(n_drones=M, reset_center=[0, 0, 1], form_center=[0, 0, 1], **BASE)
    a = np.full((M, 4), HOVER, dtype=np.float32)
    t0 = env.targets.copy()
    for _ in range(10):
        env.step(a)
    assert np.array_equal(env.targets, t0)
    over = dict(BASE, episode_len_s=0.5, auto_reset=1)
    env, _ = make_env(n_drones=M, form_path_n=4, form_path=SQUARE, form_speed=0.5, reset_center=[0, 0, 1], **over)
    for k in range(24):
        env.step(a)
    assert env.outputs()[2][0] == 2 and np.allclose(centre_of(env, M)[0], [0, 0, 1], atol=1e-12)      # truncated: new episode at vertex 0
    env.step(a)
    assert np.allclose(centre_of(env, M)[0], [0.5 / 48, 0, 1], atol=1e-12)
