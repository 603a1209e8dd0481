"""Pins of the oracle's latency rows of Table 4 ("action latency U[0, 50] ms (per ep.)", "sensor latency
U[0, 20] ms (per ep.)"; reading Q51: delays quantised to physics substeps).  Expected values are closed forms of vertical
flight under piecewise-constant thrust and of free fall, a shift-equivalence invariant for the controller action types, and
the uniform distribution of the delays; none comes from the oracle or the CUDA path."""
import math

import numpy as np
import pytest
from scipy import stats

from oracle import oracle as O
from oracle_util import FREE, make_env, set_state
from paper_2606_08039_b200 import workloads as W

M_, G_, KF = 0.027, 9.81, 3.16e-10
H = 1.0 / 240.0
K = 5
N0 = float(W.hover_rpm_f32())
N1 = float(np.float32(1.1 * N0))


def z_after_thrust_step(d, s0, steps, z0=1.0):
    """Altitude and climb rate after `steps` control steps when the rotor command changes from N0 to N1 in the row issued at
    control step s0 and that row takes effect d substeps later: constant acceleration a0, then a1."""
    a0, a1 = 4 * KF * N0 * N0 / M_ - G_, 4 * KF * N1 * N1 / M_ - G_
    t1 = min(s0 * K + d, steps * K) * H
    t2 = steps * K * H - t1
    v1 = a0 * t1
    return z0 + 0.5 * a0 * t1 * t1 + v1 * t2 + 0.5 * a1 * t2 * t2, v1 + a1 * t2


def thrust_step_run(n_envs, s0, steps, **over):
    env, _ = make_env(n_envs=n_envs, reset_center=[0, 0, 1.0], reset_half=[0, 0, 0], **over, **FREE)
    env.reset(11)
    for t in range(steps):
        env.step(np.full((n_envs, 4), N0 if t < s0 else N1, dtype=np.float32))
    return env


@pytest.mark.parametrize("d", [0, 1, 2, 4, 5, 6, 9, 10, 11, 12])
def test_rotor_command_takes_effect_d_substeps_after_it_is_issued(d):
    tau = d / 240.0
    env = thrust_step_run(1, s0=2, steps=6, act_latency_lo=tau, act_latency_hi=tau)
    z, vz = z_after_thrust_step(d, 2, 6)
    assert abs(env.state[0, 2] - z) < 1e-12 and abs(env.state[0, 9] - vz) < 1e-12, (d, env.state[0, 2], z)
    assert abs(z - z_after_thrust_step(d + 1, 2, 6)[0]) > 1e-6        # one substep more is visible at this tolerance


def test_delays_are_uniform_over_the_substep_range_and_drawn_per_episode():
    N = 6500
    env = thrust_step_run(N, s0=2, steps=6, act_latency_lo=0.0, act_latency_hi=0.050)       # Table 4: U[0, 50] ms -> 0..12 substeps
    table = np.array([z_after_thrust_step(d, 2, 6)[0] for d in range(13)])
    err = np.abs(env.state[:, 2][:, None] - table[None, :])
    d_of = err.argmin(axis=1)
    assert err.min(axis=1).max() < 1e-12                                # every env follows one of the 13 closed forms
    counts = np.bincount(d_of, minlength=13)
    assert stats.chisquare(counts).pvalue > 1e-3, counts
    # another episode draws again: truncation after 6 steps, same protocol in the second episode
    env2, _ = make_env(n_envs=N, reset_center=[0, 0, 1.0], reset_half=[0, 0, 0], act_latency_lo=0.0, act_latency_hi=0.050,
                       term_mode=W.TERM_NONE, auto_reset=1, episode_len_s=6 / 48)
    env2.reset(11)
    for ep in range(2):
        for t in range(6):
            if ep == 1 and t == 5:
                break                                                   # look before the second truncation resets the state
            env2.step(np.full((N, 4), N0 if t < 2 else N1, dtype=np.float32))
    table5 = np.array([z_after_thrust_step(d, 2, 5)[0] for d in range(13)])
    err2 = np.abs(env2.state[:, 2][:, None] - table5[None, :])
    assert err2.min(axis=1).max() < 1e-12
    d2 = err2.argmin(axis=1)
    assert abs(np.corrcoef(d_of, d2)[0, 1]) < 5 / math.sqrt(N) and stats.chisquare(np.bincount(d2, minlength=13)).pvalue > 1e-3


@pytest.mark.parametrize("act,d", [(W.ACT_VEL, 3), (W.ACT_VEL, 5), (W.ACT_VEL, 6), (W.ACT_PID, 12), (W.ACT_ATTITUDE, 8), (W.ACT_RPM, 10)])
def test_whole_step_latency_equals_the_shifted_action_sequence(act, d):
    """A controller decodes once per control step from the row that has arrived: latency d means the row of ceil(d / K) steps
    ago (the episode's first row until then).  For direct rotor commands the same holds when d is a multiple of K."""
    n = -(-d // K)
    rng = np.random.default_rng(3)
    if act == W.ACT_RPM:
        seq = (N0 * rng.uniform(0.9, 1.1, (14, 1, 4))).astype(np.float32)
    elif act == W.ACT_PID:
        seq = rng.uniform([-0.5, -0.5, 0.8, -0.3], [0.5, 0.5, 1.2, 0.3], (14, 1, 4)).astype(np.float32)
    else:
        seq = rng.uniform(-0.3, 0.3, (14, 1, 4)).astype(np.float32)
    lat, _ = make_env(action=act, act_latency_lo=d / 240.0, act_latency_hi=d / 240.0, **FREE)
    ref, _ = make_env(action=act, **FREE)
    for env in (lat, ref):
        env.reset(4)
    for t in range(14):
        lat.step(seq[t])
        ref.step(seq[max(t - n, 0)])
        assert np.array_equal(lat.state, ref.state) and np.array_equal(lat.pid, ref.pid), t
    assert np.abs(lat.state[0, 0:3] - [0, 0, 1]).max() > 1e-3             # the drone did move


def test_sensors_report_the_state_d_substeps_ago_in_free_fall():
    """Zero rotor speed from rest at z0: z = z0 - g t^2 / 2, v_z = -g t (PAPER.md:106-113 in its simplest case); the row after
    control step s with sensor latency d shows t = (s K - d) h while the state itself is at t = s K h."""
    z0 = 2.5
    for d in range(6):
        tau = d / 240.0
        env, _ = make_env(reset_center=[0, 0, z0], reset_half=[0, 0, 0], obs_latency_lo=tau, obs_latency_hi=tau, **FREE)
        env.reset(2)
        for s in (1, 2, 3):
            env.step(np.zeros((1, 4), dtype=np.float32))
            obs = env.outputs()[0][0]
            ts, tt = (s * K - d) * H, s * K * H
            assert abs(obs[2] - (z0 - 0.5 * G_ * ts * ts)) < 1e-12 and abs(obs[8] + G_ * ts) < 1e-12, (d, s)
            assert abs(env.state[0, 2] - (z0 - 0.5 * G_ * tt * tt)) < 1e-12 and abs(env.state[0, 9] + G_ * tt) < 1e-12
    # attitude is delayed with the rest of the row: constant yaw rate, quaternion and yaw angle of the KIN20 row
    env, _ = make_env(obs_mode=W.OBS_KIN20, obs_latency_lo=2 / 240.0, obs_latency_hi=2 / 240.0, **FREE)
    env.reset(2)
    set_state(env, p=[0, 0, 1], q=[1, 0, 0, 0], v=[0, 0, 0], w=[0, 0, 0.8])
    a = np.full((1, 4), N0, dtype=np.float32)
    env.step(a)
    obs = env.outputs()[0][0]
    psi = 0.8 * 3 * H                                                   # three of the five substeps
    assert abs(obs[9] - psi) < 1e-9 and abs(obs[3] - math.cos(psi / 2)) < 1e-9 and abs(obs[6] - math.sin(psi / 2)) < 1e-9
    assert np.array_equal(obs[16:20], a[0].astype(np.float64))           # the issued row


def test_sensor_delays_are_uniform_per_episode_and_the_reset_row_is_undelayed():
    N, z0 = 6000, 2.5
    env, _ = make_env(n_envs=N, reset_center=[0, 0, z0], reset_half=[0, 0, 0], obs_latency_lo=0.0, obs_latency_hi=0.020,   # Table 4: U[0, 20] ms
                      term_mode=W.TERM_NONE, auto_reset=1, episode_len_s=3 / 48)
    env.reset(6)
    zero = np.zeros((N, 4), dtype=np.float32)
    env.step(zero)
    table = np.array([z0 - 0.5 * G_ * ((K - d) * H) ** 2 for d in range(6)])
    err = np.abs(env.outputs()[0][:, 2][:, None] - table[None, :])
    assert err.min(axis=1).max() < 1e-12
    d1 = err.argmin(axis=1)
    assert stats.chisquare(np.bincount(d1, minlength=6)).pvalue > 1e-3      # round(0.020 * 240) = 5: delays 0..5
    env.step(zero); env.step(zero)                                        # truncation: the row is the new episode's initial state
    obs, _, done, _ = env.outputs()
    assert (done == 2).all() and np.array_equal(obs[:, 2], np.full(N, z0)) and np.array_equal(obs[:, 8], np.zeros(N))
    env.step(zero)
    err = np.abs(env.outputs()[0][:, 2][:, None] - table[None, :])
    assert err.min(axis=1).max() < 1e-12
    d2 = err.argmin(axis=1)
    assert abs(np.corrcoef(d1, d2)[0, 1]) < 5 / math.sqrt(N)              # drawn again for the second episode


def test_latency_ranges_outside_the_supported_window_are_rejected():
    for over in (dict(act_latency_lo=0.0, act_latency_hi=0.070), dict(obs_latency_lo=0.0, obs_latency_hi=0.030),
                 dict(act_latency_lo=0.02, act_latency_hi=0.01)):
        with pytest.raises(ValueError):
            make_env(**over, **FREE)
