"""Pins of the oracle's action decode, PID, wind, RNG and env epilogue (SURVEY.md §8(c) "Pins").

Expected values: published Philox known answers (tests/golden/), closed forms, an independent
3-state linear recurrence, statistics of the stationary AR(1) process, and hand-built states.
"""
import os

import numpy as np
import pytest
from scipy import stats
from scipy.spatial.transform import Rotation

from oracle import oracle as O
from oracle_util import FREE, GOLDEN, make_env, quat_wxyz_from_scipy, set_state
from paper_2606_08039_b200 import workloads as W


# ---- O12 Philox ----------------------------------------------------------------------------------
def test_philox_known_answers():
    n = 0
    with open(os.path.join(GOLDEN, "philox4x32_10_kat.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            w = [int(x, 16) for x in line.split()]
            assert list(O.philox(w[0:4], w[4:6])) == w[6:10]
            n += 1
    assert n == 3


def test_harness_actions_are_philox_stream3_uniforms():
    """a = base * fma(hi - lo, u, lo), u = (x >> 8) 2^-24, counter (env, drone, t, 3), key = seed halves."""
    seed, t, N, M = (5 << 32) | 77, 9, 3, 2
    a = O.gen_actions(seed, t, N, M, 100.0, 0.9, 1.1)
    assert a.dtype == np.float32 and a.shape == (N * M, 4)
    for e in range(N):
        for i in range(M):
            x = O.philox([e, i, t, 3], [77, 5])
            u = (x >> 8).astype(np.float64) / 2 ** 24
            lo, hi = np.float32(0.9), np.float32(1.1)
            ref = np.float32(100.0) * (np.float64(hi - lo) * u + np.float64(lo)).astype(np.float32)
            assert np.array_equal(a[e * M + i], ref.astype(np.float32))
    big = O.gen_actions(1, 0, 4096, 4, 1.0, -1.0, 1.0).ravel()
    assert big.min() >= -1 and big.max() < 1
    assert stats.kstest((big + 1) / 2, "uniform").pvalue > 1e-3


# ---- O3 PID -------------------------------------------------------------------------------------
def test_allocation_round_trip():
    """Random wrench -> per-rotor thrusts -> Eq.1-3 wrench, <= 1e-15 relative (SURVEY pin O3)."""
    P = O.OracleParams()
    rng = np.random.default_rng(3)
    for _ in range(200):
        T = rng.uniform(0.1, 0.5)
        tau = rng.normal(size=3) * [2e-3, 2e-3, 2e-3]
        s = O.alloc_inverse(P, T, tau)
        rpm = np.sqrt(np.abs(s) / 3.16e-10)
        if (s < 0).any():
            continue
        T2, tau2, _ = O.motor_wrench(P, rpm)
        assert abs(T2 - T) < 1e-14 * T and np.abs(tau2 - tau).max() < 1e-14 * max(1e-3, np.abs(tau).max())


def test_pid_fixed_point_is_hover_rpm():
    """p = p*, v = 0, level: every rotor at HOVER_RPM (SURVEY pin O3)."""
    for act, a in ((W.ACT_PID, [0.3, -0.2, 1.1, 0.0]), (W.ACT_VEL, [0, 0, 0, 0])):
        env, P = make_env(action=act, **FREE)
        set_state(env, p=[0.3, -0.2, 1.1], q=[1, 0, 0, 0], v=[0, 0, 0], w=[0, 0, 0])
        rpm = env.probe_decode(np.array(a, dtype=np.float32))
        # the fp32 action rounds the waypoint by <= 6e-8 m, so the fixed point holds to ~1e-8 relative
        assert np.abs(rpm / P.derived()["hover_rpm"] - 1).max() < 1e-7


def test_pid_level_z_axis_is_an_exact_linear_recurrence():
    """Level, x = y = 0 error: T = m a*_z, so z follows an independent 3-state recurrence (z, vz, Iz)
    at substep granularity (SURVEY pin O3).  Integral clamp exercised by a far waypoint."""
    for ztgt, steps in ((1.5, 96), (2.5, 200)):
        env, P = make_env(action=W.ACT_PID, **FREE)
        set_state(env, p=[0, 0, 1.0], q=[1, 0, 0, 0], v=[0, 0, 0], w=[0, 0, 0])
        pm = env.pid; pm[0, 6:10] = [0, 0, 1.0, 0]; env.pid = pm
        z, vz, Iz = 1.0, 0.0, 0.0
        h, dtc, m, g = 1 / 240, 1 / 48, 0.027, 9.81
        smax4 = 4 * P.derived()["s_max"]
        saw_clamp = False
        for _ in range(steps):
            env.step(np.array([0, 0, ztgt, 0], dtype=np.float32))
            e = ztgt - z
            Iz = min(max(Iz + e * dtc, -2.0), 2.0)
            saw_clamp |= abs(Iz) == 2.0
            acc = 1.0 * e + 0.01 * Iz + 2.0 * (0 - vz) + g
            T = min(max(m * abs(acc), 0.0), smax4)
            a = T / m - g
            for _ in range(5):
                z += h * vz + 0.5 * h * h * a
                vz += h * a
            s = env.state[0]
            assert abs(s[2] - z) < 1e-10 and abs(s[9] - vz) < 1e-10
            assert abs(env.pid[0, 2] - Iz) < 1e-12
            assert np.abs(s[[0, 1, 4, 5, 6, 10, 11, 12]]).max() < 1e-14
        assert saw_clamp == (ztgt == 2.5)


def test_pid_clamps_and_signs_on_hand_built_states():
    env, P = make_env(action=W.ACT_PID, **FREE)
    d = P.derived()
    # far waypoint in +x: pitch target saturates at +tilt_max, tau_y clamps at +tau_xy_max
    set_state(env, p=[0, 0, 1.0], q=[1, 0, 0, 0], v=[0, 0, 0], w=[0, 0, 0])
    rpm = env.probe_decode(np.array([15.0, 0, 1.0, 0], dtype=np.float32))
    T, tau, _ = O.motor_wrench(P, rpm[0])
    assert abs(tau[1] - min(P.get("tau_xy_max"), 2e-3 * 0.5)) < 1e-12 and abs(tau[0]) < 1e-15
    # +y error -> negative roll torque (R_x(phi) z = (0, -sin phi, cos phi))
    rpm = env.probe_decode(np.array([0, 15.0, 1.0, 0], dtype=np.float32))
    _, tau, _ = O.motor_wrench(P, rpm[0])
    assert tau[0] < 0 and abs(tau[1]) < 1e-15
    # yaw error -> positive tau_z, clamped
    rpm = env.probe_decode(np.array([0, 0, 1.0, 3.0], dtype=np.float32))
    _, tau, _ = O.motor_wrench(P, rpm[0])
    assert abs(tau[2] - min(P.get("tau_z_max"), 1e-3 * 3.0)) < 1e-9
    # thrust saturates at 4 s_max for a waypoint far above
    rpm = env.probe_decode(np.array([0, 0, 500.0, 0], dtype=np.float32))
    assert np.allclose(rpm, d["max_rpm"], rtol=1e-12)
    # D term acts on the measured body rate with a minus sign
    set_state(env, w=[1.0, 0, 0])
    rpm = env.probe_decode(np.array([0, 0, 1.0, 0], dtype=np.float32))
    _, tau, _ = O.motor_wrench(P, rpm[0])
    assert abs(tau[0] + 5e-4) < 1e-12


def test_dsl_setpoint_rate_limits():
    """held setpoint moves at most 2.0 m/s and pi rad/s; integral clamps halved."""
    env, P = make_env(action=W.ACT_PID, dsl=1, int_clamp_pos=1.0, int_clamp_att=0.25, **FREE)
    set_state(env, p=[0, 0, 1.0], q=[1, 0, 0, 0], v=[0, 0, 0], w=[0, 0, 0])
    pm = env.pid; pm[0, 6:10] = [0, 0, 1.0, 0]; env.pid = pm
    a = np.array([3.0, 4.0, 1.0, 2.0], dtype=np.float32)
    env.probe_decode(a, commit=True)
    sp = env.pid[0, 6:10]
    assert np.allclose(sp[:3], [0.6 * 2 / 48, 0.8 * 2 / 48, 1.0], atol=1e-15) and abs(sp[3] - np.pi / 48) < 1e-15
    for _ in range(200):
        env.probe_decode(a, commit=True)
    sp = env.pid[0, 6:10]
    assert np.allclose(sp, [3, 4, 1, 2], atol=1e-12)
    assert abs(env.pid[0, 0:3]).max() <= 1.0 and abs(env.pid[0, 3:6]).max() <= 0.25


def test_vel_action_heading_frame():
    """Q20: VEL = [vx, vy, vz, wz] in the yaw-only heading frame; position error zero, I_p frozen."""
    env, P = make_env(action=W.ACT_VEL, **FREE)
    yaw = 0.7
    q = quat_wxyz_from_scipy(Rotation.from_euler("z", yaw))
    v_world = Rotation.from_euler("z", yaw).apply([0.4, -0.3, 0.2])
    set_state(env, p=[1, 2, 1.0], q=q, v=v_world, w=[0, 0, 0])
    rpm = env.probe_decode(np.array([0.4, -0.3, 0.2, 0.0], dtype=np.float32), commit=True)
    assert np.abs(rpm / P.derived()["hover_rpm"] - 1).max() < 1e-7   # already tracking: hover thrust
    assert np.abs(env.pid[0, 0:3]).max() == 0.0
    rpm = env.probe_decode(np.array([0.4, -0.3, 0.2, 1.0], dtype=np.float32))
    _, tau, _ = O.motor_wrench(P, rpm[0])
    assert abs(tau[2] - (1e-3 * (1.0 / 48) + 1e-4 * (1.0 / 48) ** 2)) < 1e-12 and abs(tau[0]) < 1e-9 and abs(tau[1]) < 1e-9   # fp32 actions round 0.4, -0.3


def test_pid_closed_loop_reaches_waypoint():
    """Sanity of the reading (SURVEY feasibility probe): a CF2X flies to a waypoint 1.2 m away and stays
    far inside config 3's 0.4 rad limit.  Not a numeric pin."""
    env, _ = make_env(action=W.ACT_PID, dsl=1, int_clamp_pos=1.0, int_clamp_att=0.25, **FREE)
    set_state(env, p=[0, 0, 1.0], q=[1, 0, 0, 0], v=[0, 0, 0], w=[0, 0, 0])
    pm = env.pid; pm[0, 6:10] = [0, 0, 1.0, 0]; env.pid = pm
    tgt = np.array([0.8, -0.6, 1.65, 0], dtype=np.float32)
    tilt = 0.0
    for _ in range(480):
        env.step(tgt)
        tilt = max(tilt, np.abs(O.euler_zyx(env.state[0, 3:7])[:2]).max())
    assert np.linalg.norm(env.state[0, 0:3] - tgt[:3]) < 0.1 and tilt < 0.1


# ---- O9 wind --------------------------------------------------------------------------------------
def test_wind_ar1_statistics_and_force_law():
    """x <- a x + sigma sqrt(1 - a^2) xi (Q27): stationary variance sigma^2, lag-k
    autocorrelation a^k; F = k_w |w - v| (w - v) (Q28)."""
    N = 8192
    env, P = make_env(n_envs=N, physics=W.PHYS_MJC, aero_mask=W.AERO_WIND, threads=8, **FREE)
    alpha = np.exp(-(1 / 48) / 1.0)
    hist = []
    a = np.zeros((N, 4), dtype=np.float32)
    for t in range(400):
        env.step(a)
        if t >= 250:
            hist.append(env.wind.copy())
    hist = np.array(hist)                                              # [T, N, 3]
    var = hist.var(axis=(0, 1))
    assert np.abs(var / 0.25 - 1).max() < 0.03
    for k in (1, 10, 48):
        c = (hist[k:] * hist[:-k]).mean(axis=(0, 1)) / (hist * hist).mean(axis=(0, 1))
        assert np.abs(c - alpha ** k).max() < 0.03
    # components independent, normals standard
    xi = np.array([O.wind_normals(3, e, 1) for e in range(4000)])
    assert stats.kstest(xi.ravel(), "norm").pvalue > 1e-3
    assert np.abs(np.corrcoef(xi.T) - np.eye(3)).max() < 0.06
    # force law with w = 0: F = -k_w |v| v on top of the rotor force
    env1, P1 = make_env(aero_mask=W.AERO_WIND, **FREE)
    v = np.array([1.0, -2.0, 0.5])
    set_state(env1, p=[0, 0, 5], q=[1, 0, 0, 0], v=v, w=[0, 0, 0])
    F, _ = env1.probe_wrench(0, [0, 0, 0, 0])
    assert np.allclose(F[0], -6.125e-3 * np.linalg.norm(v) * v, rtol=1e-12)
    env1.wind = [[0.3, 0.1, -0.2]]
    F, _ = env1.probe_wrench(0, [0, 0, 0, 0])
    rel = np.array([0.3, 0.1, -0.2]) - v
    assert np.allclose(F[0], 6.125e-3 * np.linalg.norm(rel) * rel, rtol=1e-12)


def test_wind_is_updated_once_per_control_step_with_the_documented_draw():
    env, P = make_env(aero_mask=W.AERO_WIND, **FREE)
    env.reset(42)
    env.step(np.zeros(4))
    alpha = np.exp(-1 / 48)
    assert np.allclose(env.wind[0], 0.5 * np.sqrt(1 - alpha ** 2) * O.wind_normals(42, 0, 1), rtol=1e-12)
    w1 = env.wind[0].copy()
    env.step(np.zeros(4))
    assert np.allclose(env.wind[0], alpha * w1 + 0.5 * np.sqrt(1 - alpha ** 2) * O.wind_normals(42, 0, 2), rtol=1e-12)


# ---- O10 observation / reward / termination on hand-built states ---------------------------------------
def _one_step_outputs(state_rows, targets=None, rpm=None, n_drones=1, **over):
    env, P = make_env(n_drones=n_drones, auto_reset=0, **over)
    s = env.state
    s[:] = np.asarray(state_rows, dtype=float).reshape(n_drones, 13)
    env.state = s
    if targets is not None:
        env.targets = np.asarray(targets, dtype=float).reshape(n_drones, 4)
    kf = 0.027 * 9.81 / (4 * 16384.0 ** 2)
    a = np.full((n_drones, 4), 16384.0 if rpm is None else rpm, dtype=np.float32)
    env.step(a)
    return env, kf


def test_hover_reward_eq8_and_termination_rules():
    """Eq.8 and the termination rule of PAPER.md:309 on states at rest at hover thrust
    (k_f chosen so hover RPM is exactly 16384 -> the state does not move during the step)."""
    kf = 0.027 * 9.81 / (4 * 16384.0 ** 2)
    base = dict(k_f=kf, reward_mode=W.REW_HOVER, term_mode=W.TERM_HOVER)
    lvl = [1, 0, 0, 0]
    cases = [
        ([0.3, -0.4, 1.2], lvl, -0.2 - 0.1 * 0.5, 0),
        ([0.0, 0.0, 1.0], lvl, 0.5, 0),                                # at target
        ([0.03, 0.0, 1.03], lvl, -0.03 - 0.003 + 0.5, 0),              # inside the 0.05 m ball
        ([0.03, 0.03, 1.03], lvl, -0.03 - 0.1 * np.hypot(0.03, 0.03), 0),   # |d| = 0.052: outside
    ]
    for p, q, r_ref, d_ref in cases:
        env, _ = _one_step_outputs(p + q + [0] * 6, **base)
        obs, rew, done, _ = env.outputs()
        assert abs(rew[0] - r_ref) < 1e-12 and done[0] == d_ref, (p, rew[0], r_ref)
        assert np.allclose(obs[0], p + [0, 0, 0] + [0] * 6, atol=1e-12)
    # z > 3 m terminates without the crash penalty (Q24)
    env, _ = _one_step_outputs([0, 0, 3.5] + lvl + [0] * 6, **base)
    _, rew, done, _ = env.outputs()
    assert done[0] == 1 and abs(rew[0] + 2.5) < 1e-12
    env, _ = _one_step_outputs([0, 0, 2.999] + lvl + [0] * 6, **base)
    assert env.outputs()[2][0] == 0
    # roll beyond pi/2 terminates with the crash penalty; velocity and tilt terms of Eq.8
    q = quat_wxyz_from_scipy(Rotation.from_euler("x", 1.7))
    env, _ = _one_step_outputs([0, 0, 50.0] + list(q) + [0] * 6, rpm=0.0, **base)
    obs, rew, done, _ = env.outputs()
    vz = -9.81 / 48
    assert done[0] == 1
    assert abs(rew[0] - (-abs(obs[0, 2] - 1) - 0.05 * abs(vz) - 0.05 * 1.7 - 100)) < 1e-9
    assert abs(obs[0, 3] - 1.7) < 1e-12 and abs(obs[0, 8] - vz) < 1e-12


def test_config3_reward_and_termination():
    kf = 0.027 * 9.81 / (4 * 16384.0 ** 2)
    base = dict(k_f=kf, reward_mode=W.REW_NEG_SQ_DIST, term_mode=W.TERM_TILT_DIST, term_tilt=0.4)
    env, _ = _one_step_outputs([0.5, 0.5, 1.0, 1, 0, 0, 0] + [0] * 6, targets=[1, -1, 2, 0], **base)
    _, rew, done, _ = env.outputs()
    assert abs(rew[0] + (0.25 + 2.25 + 1.0)) < 1e-12 and done[0] == 0
    env, _ = _one_step_outputs([2.0, 2.0, 1.1, 1, 0, 0, 0] + [0] * 6, targets=[0, 0, 1, 0], **base)
    assert env.outputs()[2][0] == 1                                    # |p| = 3.04 > 3
    env, _ = _one_step_outputs([2.0, 2.0, 0.9, 1, 0, 0, 0] + [0] * 6, targets=[0, 0, 1, 0], **base)
    assert env.outputs()[2][0] == 0                                    # |p| = 2.97
    for ang, d_ref in ((0.39, 0), (0.41, 1)):
        q = quat_wxyz_from_scipy(Rotation.from_euler("y", -ang))
        env, _ = _one_step_outputs([0, 0, 1.0] + list(q) + [0] * 6, rpm=0.0, **base)
        assert env.outputs()[2][0] == d_ref


def test_formation_reward_adjacency_and_multi_hover_sum():
    kf = 0.027 * 9.81 / (4 * 16384.0 ** 2)
    M = 3
    pos = np.array([[0.3, 0, 1.0], [-0.1, 0.3, 1.1], [-0.2, -0.2, 0.9]])
    slots = np.array([[0.3, 0, 1.0], [-0.15, 0.2598, 1.0], [-0.15, -0.2598, 1.0]])
    rows = [list(p) + [1, 0, 0, 0] + [0] * 6 for p in pos]
    tg = [list(s) + [0] for s in slots]
    env, _ = _one_step_outputs(rows, targets=tg, n_drones=M, k_f=kf, reward_mode=W.REW_FORMATION,
                               term_mode=W.TERM_FORMATION, obs_mode=W.OBS_KIN12_ADJ, adj_radius=0.45,
                               term_center=[0, 0, 1])
    obs, rew, done, margin = env.outputs()
    r = -sum(np.linalg.norm(pos[i] - slots[i]) for i in range(M))
    for i in range(M):
        for j in range(i + 1, M):
            r -= 0.5 * abs(np.linalg.norm(pos[i] - pos[j]) - np.linalg.norm(slots[i] - slots[j]))
    assert abs(rew[0] - r) < 1e-12 and done[0] == 0
    o = obs[0].reshape(M, 12 + M)
    dist = np.linalg.norm(pos[:, None] - pos[None], axis=-1)
    assert np.array_equal(o[:, 12:], (dist < 0.45).astype(float))      # diagonal 1 (Q23)
    assert abs(margin[0, 2] - np.abs(dist[dist > 0] - 0.45).min()) < 1e-12
    assert np.allclose(o[:, 0:3], pos, atol=1e-12)
    # multi-hover: sum of per-drone Eq.8 with per-drone targets
    env, _ = _one_step_outputs(rows, targets=tg, n_drones=M, k_f=kf, reward_mode=W.REW_MULTI_HOVER, term_mode=W.TERM_HOVER)
    _, rew, _, _ = env.outputs()
    r = sum(-abs(pos[i, 2] - slots[i, 2]) - 0.1 * np.hypot(*(pos[i, :2] - slots[i, :2])) + (0.5 if np.linalg.norm(pos[i] - slots[i]) < 0.05 else 0) for i in range(M))
    assert abs(rew[0] - r) < 1e-12


# ---- reset distribution, auto-reset, truncation ----------------------------------------------------------
def test_reset_distributions_of_the_five_configs():
    for c in range(1, 6):
        wl = W.config(c)
        N = min(wl.n_envs, 2048)
        P = O.OracleParams(0, **wl.params)
        env = O.OracleEnv(N, wl.n_drones, wl.physics_mode, wl.action_type, P)
        env.reset(wl.seed)
        s = env.state.reshape(N, wl.n_drones, 13)
        assert np.all(s[..., 3] == 1) and np.all(s[..., 4:] == 0)
        p = s[..., 0:3]
        tg = env.targets.reshape(N, wl.n_drones, 4)
        if c in (1, 3):
            assert np.abs(p - [0, 0, 1]).max() <= 0.1
        if c == 2:
            assert np.all(p[..., :2] == 0) and p[..., 2].min() >= 0.05 and p[..., 2].max() < 1.5
            assert stats.kstest((p[..., 2].ravel() - 0.05) / 1.45, "uniform").pvalue > 1e-3
        if c == 3:
            assert (tg[..., :3] >= [-1, -1, 0.2]).all() and (tg[..., :3] < [1, 1, 2.0]).all()
            assert stats.kstest((tg[..., 2].ravel() - 0.2) / 1.8, "uniform").pvalue > 1e-3
        if c == 4:
            gx = (np.arange(8) % 4 - 1.5) * 0.3
            gy = (np.arange(8) // 4 - 0.5) * 0.3
            assert np.abs(p[..., 0] - gx).max() <= 0.05 and np.abs(p[..., 1] - gy).max() <= 0.05
            assert p[..., 2].min() >= 0.3 and p[..., 2].max() < 1.2
            assert np.allclose(tg[..., 2], np.linspace(0.7, 1.2, 8)) and np.array_equal(tg[..., :2], p[..., :2])
        if c == 5:
            ang = 2 * np.pi * np.arange(4) / 4
            slots = np.stack([0.3 * np.cos(ang), 0.3 * np.sin(ang), np.ones(4)], -1)
            assert np.abs(p - slots).max() <= 0.05 and np.allclose(tg[..., :3], slots, atol=1e-15)
        if c in (1, 2):
            assert np.all(tg == [0, 0, 1, 0])
        # a bigger batch draws the same values for the same env (counter-based: partition independent)
        env2 = O.OracleEnv(N // 2 + 1, wl.n_drones, wl.physics_mode, wl.action_type, P)
        env2.reset(wl.seed)
        assert np.array_equal(env2.state, env.state[: (N // 2 + 1) * wl.n_drones])


def test_auto_reset_and_truncation_semantics():
    """Q29: reward/done describe the finished transition, obs opens the new episode; truncation at the
    episode length (Table 5)."""
    env, P = make_env(n_envs=3, episode_len_s=0.125, auto_reset=1, term_mode=W.TERM_HOVER)
    env.reset(9)
    n = P.derived()["hover_rpm"]
    a = np.full((3, 4), n, dtype=np.float32)
    a[1] = 0.0                                                         # env 1 falls: 1 m takes 0.45 s
    first = env.state.copy()
    for t in range(1, 7):
        env.step(a)
        obs, rew, done, _ = env.outputs()
        if t < 6:
            assert not done.any() and np.array_equal(env.ep_step, [t] * 3)
    assert list(done) == [2, 2, 2]                                     # 0.125 s * 48 Hz = 6 steps
    assert np.array_equal(env.ep_step, [0, 0, 0])
    s = env.state
    assert np.all(s[:, 3] == 1) and np.all(s[:, 7:] == 0) and not np.array_equal(s, first)
    assert np.allclose(obs[:, 0:3], s[:, 0:3]) and np.all(obs[:, 3:] == 0)
    # reward of the finished transition: env 1 fell freely for 0.125 s from its first spawn point
    z = first[1, 2] - 0.5 * 9.81 * 0.125 ** 2
    r_ref = -abs(z - 1) - 0.1 * np.hypot(first[1, 0], first[1, 1]) - 0.05 * 9.81 * 0.125
    r_ref += 0.5 if np.linalg.norm([first[1, 0], first[1, 1], z - 1]) < 0.05 else 0.0
    assert abs(rew[1] - r_ref) < 1e-12
    # floor crash resets only that env, at the global step index
    env, P = make_env(n_envs=2, auto_reset=1, term_mode=W.TERM_HOVER)
    env.reset(9)
    a = np.full((2, 4), n, dtype=np.float32); a[1] = 0.0
    for t in range(1, 40):
        env.step(a)
        _, rew, done, _ = env.outputs()
        if done[1]:
            break
    assert done[1] == 1 and done[0] == 0 and rew[1] < -100 and env.ep_step[1] == 0 and env.ep_step[0] == t
    x = O.philox([1, 0, t, 0], [9, 0])
    assert abs(env.state[1, 0] - (-0.1 + 0.2 * (x[0] >> 8) / 2 ** 24)) < 1e-15


def test_threads_do_not_change_results():
    wl = W.config(5).scaled(64)
    P = O.OracleParams(0, **wl.params)
    outs = []
    for th in (1, 4):
        env = O.OracleEnv(wl.n_envs, wl.n_drones, wl.physics_mode, wl.action_type, P, n_threads=th)
        env.reset(wl.seed)
        for t in range(5):
            env.step(O.gen_actions(wl.seed, t, wl.n_envs, wl.n_drones, 1.0, -1.0, 1.0))
        outs.append((env.state, env.outputs()[0]))
    assert np.array_equal(outs[0][0], outs[1][0]) and np.array_equal(outs[0][1], outs[1][1])


def test_flop_tally_is_positive_and_state_preserving():
    wl = W.config(5).scaled(8)
    P = O.OracleParams(0, **wl.params)
    env = O.OracleEnv(wl.n_envs, wl.n_drones, wl.physics_mode, wl.action_type, P)
    env.reset(wl.seed)
    a = O.gen_actions(wl.seed, 0, wl.n_envs, wl.n_drones, 1.0, -1.0, 1.0)
    s0 = env.state.copy()
    f = env.flop_tally(a)
    assert np.array_equal(env.state, s0)
    per_drone = f / (wl.n_envs * wl.n_drones)
    assert 2000 < per_drone < 8000, per_drone
