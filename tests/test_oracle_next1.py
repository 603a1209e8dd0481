"""Pins of the oracle's SURVEY.md §8(f) NEXT-1 parts: normalised RPM actions, ONE_D_RPM, ATTITUDE, the 20-dim KIN
observation and the +-configuration (CF2P) mixing.  Expected values come from the paper's statements and from
closed forms worked out here, never from the oracle or the CUDA path."""
import math

import numpy as np

from oracle import oracle as O
from oracle_util import FREE, make_env, set_state
from paper_2606_08039_b200 import workloads as W

M, G, KF, KM, L = 0.027, 9.81, 3.16e-10, 7.94e-12, 0.0397          # Table 2, CF2X / CF2P column
JXX, JZZ = 1.4e-5, 2.17e-5
HOVER = math.sqrt(M * G / (4 * KF))
MAXR = math.sqrt(2.25 * M * G / (4 * KF))


def test_normalized_rpm_map_endpoints_and_linearity():
    """PAPER.md:300 (normalizedActionToRPM), reading Q35: -1 -> 0, 0 -> HOVER_RPM, +1 -> MAX_RPM, piecewise linear, clipped."""
    env, _ = make_env(action=W.ACT_RPM_NORM, **FREE)
    for a, want in [(-1.0, 0.0), (0.0, HOVER), (1.0, MAXR), (-0.5, 0.5 * HOVER), (0.25, HOVER + 0.25 * (MAXR - HOVER)),
                    (-7.0, 0.0), (3.0, MAXR)]:
        rpm = env.probe_decode(np.array([a, a, a, a], dtype=np.float32))
        assert np.allclose(rpm, want, rtol=1e-12, atol=1e-9), (a, rpm, want)
    rpm = env.probe_decode(np.array([-1.0, 0.0, 0.5, 1.0], dtype=np.float32))          # the four rotors are independent
    assert np.allclose(rpm[0], [0.0, HOVER, HOVER + 0.5 * (MAXR - HOVER), MAXR], rtol=1e-12)


def test_one_d_rpm_drives_all_rotors_from_the_first_component():
    env, _ = make_env(action=W.ACT_ONE_D_RPM, **FREE)
    rpm = env.probe_decode(np.array([0.5, -1.0, 1.0, 0.123], dtype=np.float32))
    assert np.allclose(rpm, HOVER + 0.5 * (MAXR - HOVER), rtol=1e-12)
    # a = 0 is hover: stationary to rounding; a > 0 is the uniform-thrust closed form z'' = 4 k_f n^2 / m - g
    set_state(env, p=[0, 0, 1.0], q=[1, 0, 0, 0], v=[0, 0, 0], w=[0, 0, 0])
    s0 = env.state.copy()
    for _ in range(48):
        env.step(np.zeros((1, 4), dtype=np.float32))
    assert np.abs(env.state - s0).max() < 1e-12
    n = HOVER + float(np.float32(0.2)) * (MAXR - HOVER)                 # the action is an fp32 number
    acc = 4 * KF * n * n / M - G
    for _ in range(48):
        env.step(np.array([[0.2, 9, 9, 9]], dtype=np.float32))
    t = 1.0
    assert abs(env.state[0, 2] - (1.0 + 0.5 * acc * t * t)) < 1e-9 and abs(env.state[0, 9] - acc * t) < 1e-9


def test_attitude_action_thrust_channel_targets_and_yaw_rate():
    """Reading Q36: [thrust (normalised map, T = 4 k_f rpm^2), roll*, pitch*, yaw rate] through the attitude loop + mixer."""
    env, P = make_env(action=W.ACT_ATTITUDE, **FREE)
    set_state(env, p=[0, 0, 1.0], q=[1, 0, 0, 0], v=[0, 0, 0], w=[0, 0, 0])
    # level, zero targets, thrust 0 -> every rotor at HOVER_RPM (no torque demanded)
    assert np.allclose(env.probe_decode(np.array([0, 0, 0, 0], dtype=np.float32)), HOVER, rtol=1e-12)
    # roll target 0.1 rad from level: tau_x = Kp * 0.1 + Ki * (0.1 dt) (Table 6: 2e-3, 0), split over the X mixer
    rpm = env.probe_decode(np.array([0, 0.1, 0, 0], dtype=np.float32))[0]
    s = KF * rpm ** 2
    l = L / math.sqrt(2)
    assert abs(l * (s[0] + s[1] - s[2] - s[3]) - 2e-3 * float(np.float32(0.1))) < 1e-12
    assert abs(s.sum() - M * G) < 1e-12 and abs(-s[0] + s[1] - s[2] + s[3]) < 1e-15
    # targets are clipped to +-tilt_max (0.5 rad)
    a = env.probe_decode(np.array([0, 5.0, 0, 0], dtype=np.float32))[0]
    b = env.probe_decode(np.array([0, 0.5, 0, 0], dtype=np.float32))[0]
    assert np.allclose(a, b, rtol=1e-14)
    # yaw rate r: psi* = psi + r dt  ->  tau_z = Kp_z r dt + Ki_z (r dt) dt  (Table 6: 1e-3, 1e-4)
    r, dt = 1.0, 1 / 48
    rpm = env.probe_decode(np.array([0, 0, 0, r], dtype=np.float32))[0]
    s = KF * rpm ** 2
    assert abs((KM / KF) * (-s[0] + s[1] - s[2] + s[3]) - (1e-3 * r * dt + 1e-4 * r * dt * dt)) < 1e-13
    # closed loop: hold roll* = 0.2 rad at hover thrust for 1 s -> settles near the target and drifts towards -y
    for _ in range(48):
        env.step(np.array([[0, 0.2, 0, 0]], dtype=np.float32))
    phi = O.euler_zyx(env.state[0, 3:7])[0]
    assert 0.15 < phi < 0.25 and env.state[0, 8] < -0.5


def test_kin20_observation_layout():
    """KIN = [p, q, eta, v, omega, a_{t-1}] (20 per drone); a_{t-1} is the action of the step that
    produced the state, zeros after reset."""
    env, _ = make_env(n_envs=2, n_drones=2, action=W.ACT_RPM, obs_mode=W.OBS_KIN20, **FREE)
    obs = env.outputs()[0].reshape(2, 2, 20)
    assert np.all(obs[:, :, 16:20] == 0.0)
    q = np.array([0.9, 0.1, -0.2, 0.3]); q /= np.linalg.norm(q)
    set_state(env, p=[0.1, -0.2, 1.3], q=q, v=[0.4, 0.5, -0.6], w=[0.7, -0.8, 0.9])
    a = (HOVER * np.array([[1.0, 1.01, 0.99, 1.02]] * 4)).astype(np.float32)
    env.step(a)
    obs = env.outputs()[0].reshape(2, 2, 20)
    st = env.state.reshape(2, 2, 13)
    assert np.array_equal(obs[:, :, 0:3], st[:, :, 0:3]) and np.array_equal(obs[:, :, 3:7], st[:, :, 3:7])
    assert np.array_equal(obs[:, :, 10:13], st[:, :, 7:10]) and np.array_equal(obs[:, :, 13:16], st[:, :, 10:13])
    for e in range(2):
        for i in range(2):
            assert np.allclose(obs[e, i, 7:10], O.euler_zyx(st[e, i, 3:7]), atol=1e-15)
    assert np.array_equal(obs[:, :, 16:20].reshape(4, 4), a.astype(np.float64))


def test_cf2p_plus_configuration_mixing():
    """PAPER.md:80, reading Q37: tau_x = L (F_1 - F_3), tau_y = L (F_2 - F_0), yaw as in the X frame; CF2X parameters."""
    P = O.OracleParams(W.MODEL_CF2P)
    assert P.get("m") == 0.027 and P.get("L") == 0.0397
    rng = np.random.default_rng(3)
    rpm = rng.uniform(0.8, 1.2, 4) * HOVER
    T, tau, _ = O.motor_wrench(P, rpm)
    F = KF * rpm ** 2
    assert abs(T - F.sum()) < 1e-15
    assert np.allclose(tau, [L * (F[1] - F[3]), L * (F[2] - F[0]), (KM / KF) * (-F[0] + F[1] - F[2] + F[3])], rtol=1e-13, atol=1e-18)
    # allocation round trip: random wrench -> per-rotor thrusts -> wrench
    for _ in range(20):
        T = rng.uniform(0.1, 0.5); tq = rng.uniform(-1, 1, 3) * [1e-3, 1e-3, 1e-4]
        s = O.alloc_inverse(P, T, tq)
        T2, tau2, _ = O.motor_wrench(P, np.sqrt(s / KF))
        assert abs(T2 - T) < 1e-14 and np.allclose(tau2, tq, rtol=1e-11, atol=1e-17)
    # pure roll torque at hover thrust: omega_x = tau_x t / J_xx exactly (principal axis, torque-free about the others)
    env, _ = make_env(model=W.MODEL_CF2P, **FREE)
    set_state(env, p=[0, 0, 1.0], q=[1, 0, 0, 0], v=[0, 0, 0], w=[0, 0, 0])
    s_h = M * G / 4
    F = np.array([s_h, 1.1 * s_h, s_h, 0.9 * s_h])
    a = np.sqrt(F / KF).astype(np.float32)[None, :]
    Fa = KF * a[0].astype(np.float64) ** 2
    for _ in range(12):
        env.step(a)
    t = 12 / 48
    assert abs(env.state[0, 10] - L * (Fa[1] - Fa[3]) * t / JXX) < 1e-9 * abs(env.state[0, 10])
    # fp32 rotor speeds leave a tiny yaw torque; it couples into omega_y only through (J_zz - J_xx) omega_z omega_x
    assert abs(env.state[0, 11]) < 1e-4 and abs(env.state[0, 12] - (KM / KF) * (-Fa[0] + Fa[1] - Fa[2] + Fa[3]) * t / JZZ) < 2e-8   # frozen world-frame torque over a substep mixes tau_y, tau_z at 9 rad/s
    # the PID default torque clamp follows the same "a third of the hover rotor thrust per axis" rule (Q17/Q37)
    assert abs(P.get("tau_xy_max") - 2 * L * s_h / 3) < 1e-15


def test_velocity_aviary_reward_target_and_observation():
    """obs [p, eta, v, omega, v*, omega_z*] (16), r = -|v - v*| - 0.1 |omega_z - omega_z*| - 0.05 (|phi| + |theta|)
    + 0.5 [tracked], target ~ U(-0.5, 0.5)^3 x U(-0.25, 0.25) per episode (reading Q38: tracked = |v - v*| < 0.05 m/s)."""
    from scipy.spatial.transform import Rotation
    from oracle_util import quat_wxyz_from_scipy
    over = dict(obs_mode=W.OBS_KIN12_TGT, reward_mode=W.REW_VELOCITY, target_mode=W.TGT_BOX, target_lo=[-0.5] * 3, target_hi=[0.5] * 3,
                target_w_lo=-0.25, target_w_hi=0.25, physics=W.PHYS_MJC)
    env, _ = make_env(n_envs=4000, **dict(over, **FREE))
    tg = env.targets
    assert np.all(np.abs(tg[:, :3]) <= 0.5) and np.all(np.abs(tg[:, 3]) <= 0.25)
    assert abs(tg[:, :3].std() - 1 / math.sqrt(12)) < 0.01 and abs(tg[:, 3].std() - 0.5 / math.sqrt(12)) < 0.005
    assert abs(np.corrcoef(tg[:, 0], tg[:, 3])[0, 1]) < 0.05 and np.abs(tg.mean(axis=0)).max() < 0.02
    obs = env.outputs()[0].reshape(4000, 16)
    assert np.array_equal(obs[:, 12:16], tg)
    # hand-built state: the reward is evaluated on the end-of-step state, so recompute it from that state
    env, _ = make_env(n_envs=1, **dict(over, **FREE))
    q = quat_wxyz_from_scipy(Rotation.from_euler("ZYX", [0.3, -0.1, 0.2]))
    set_state(env, p=[0, 0, 1.0], q=q, v=[0.3, -0.2, 0.1], w=[0.1, 0.2, -0.4])
    env.targets = np.array([[0.25, -0.1, 0.05, 0.1]])
    env.step((HOVER * np.ones((1, 4))).astype(np.float32))
    s = env.state[0]
    eta = O.euler_zyx(s[3:7])
    verr = np.linalg.norm(s[7:10] - [0.25, -0.1, 0.05])
    want = -verr - 0.1 * abs(s[12] - 0.1) - 0.05 * (abs(eta[0]) + abs(eta[1])) + (0.5 if verr < 0.05 else 0.0)
    assert abs(env.outputs()[1][0] - want) < 1e-13 and verr > 0.05
    # exactly tracked: level, at the target velocity, gravity cancelled by hover thrust -> -0 + 0.5
    set_state(env, p=[0, 0, 1.0], q=[1, 0, 0, 0], v=[0.25, -0.1, 0.05], w=[0, 0, 0])
    env.targets = np.array([[0.25, -0.1, 0.05, 0.0]])
    env.step((HOVER * np.ones((1, 4))).astype(np.float32))
    assert abs(env.outputs()[1][0] - 0.5) < 1e-6


def test_domain_randomisation_factors_draws_and_physics():
    """Table 4, reading Q39: per-episode factors U(1 - a, 1 + a) on [m, J, k_f, k_m, drag, C_gnd, C_1, g];
    each one enters the physics exactly where its nominal constant does, the controller keeps the nominal model."""
    alpha = [0.2, 0.2, 0.15, 0.15, 0.3, 0.3, 0.3, 0.02]
    env, _ = make_env(n_envs=3000, n_drones=2, dr_alpha=alpha + [0.0] * 4, **FREE)
    f = env.dr
    for a in range(8):
        assert np.all(np.abs(f[:, a] - 1.0) <= alpha[a] + 1e-12)
        assert abs(f[:, a].std() - 2 * alpha[a] / math.sqrt(12)) < 0.04 * alpha[a] and abs(f[:, a].mean() - 1.0) < 0.03 * alpha[a]
    assert np.abs(np.corrcoef(f[:, :7].T) - np.eye(7)).max() < 0.06          # independent draws
    g = f[:, 7].reshape(3000, 2)
    assert np.array_equal(g[:, 0], g[:, 1]) and not np.array_equal(f[0::2, 0], f[1::2, 0])   # g per env, vehicle factors per drone
    env0, _ = make_env(n_envs=8, n_drones=2, **FREE)
    assert np.all(env0.dr == 1.0)                                              # off by default
    # uniform thrust, level: z'' = 4 (k_f s_kf) n^2 / (m s_m) - g s_g
    env, _ = make_env(**FREE)
    sc = np.array([[1.15, 0.9, 1.1, 0.93, 1.2, 0.8, 1.25, 1.01] + [1.0] * 8])
    env.dr = sc
    set_state(env, p=[0, 0, 1.0], q=[1, 0, 0, 0], v=[0, 0, 0], w=[0, 0, 0])
    n = float(np.float32(HOVER))
    for _ in range(24):
        env.step(np.full((1, 4), n, dtype=np.float32))
    acc = 4 * KF * 1.1 * n * n / (M * 1.15) - G * 1.01
    assert abs(env.state[0, 9] - acc * 0.5) < 1e-12 and abs(env.state[0, 2] - (1.0 + 0.5 * acc * 0.25)) < 1e-12
    # pure yaw torque: omega_z = (k_m s_km) sum(+-n^2) t / (J_zz s_J)
    set_state(env, p=[0, 0, 1.0], q=[1, 0, 0, 0], v=[0, 0, 0], w=[0, 0, 0])
    a = np.array([[0.98, 1.02, 0.98, 1.02]], dtype=np.float32) * np.float32(HOVER)
    nn = a[0].astype(np.float64) ** 2
    for _ in range(12):
        env.step(a)
    want = KM * 0.93 * (-nn[0] + nn[1] - nn[2] + nn[3]) * 0.25 / (JZZ * 0.9)
    assert abs(env.state[0, 12] - want) < 1e-10 * abs(want) + 1e-13 and abs(env.state[0, 10]) < 1e-12
    # ground effect, drag and downwash coefficients scale their forces linearly (probe the substep wrench)
    envg, _ = make_env(n_drones=2, physics=W.PHYS_MJC_GND_DRAG_DW, **FREE)
    st = envg.state
    st[0, 0:3] = [0, 0, 0.1]; st[1, 0:3] = [0.05, 0, 0.6]; st[:, 7:10] = [[0.5, 0, 0], [0, 0, 0]]
    envg.state = st
    rpm = np.full((2, 4), HOVER)
    F0, _ = envg.probe_wrench(0, rpm)
    d = np.ones((2, 16)); d[0, 4:7] = [1.3, 0.7, 1.2]
    envg.dr = d
    F1, _ = envg.probe_wrench(0, rpm)
    T = M * G
    gnd = 11.36859 * T * (0.02325 / (4 * 0.1)) ** 2
    drag_x = -9.1785e-7 * 4 * (2 * math.pi * HOVER / 60) * 0.5
    dz = 0.5; dw = 2267.18 * (0.02325 / (4 * dz)) ** 2 * math.exp(-0.5 * (0.05 / (0.16 * dz - 0.11)) ** 2)
    assert abs((F1[0, 0] - F0[0, 0]) - 0.3 * drag_x) < 1e-12
    assert abs((F1[0, 2] - F0[0, 2]) - (-0.3 * gnd - 0.2 * dw)) < 1e-10
    # the controller keeps the nominal model: the PID decode of a randomised drone equals the nominal one
    envp, _ = make_env(action=W.ACT_PID, **FREE)
    r0 = envp.probe_decode(np.array([0.3, -0.2, 1.4, 0.1], dtype=np.float32))
    envp.dr = sc
    assert np.array_equal(envp.probe_decode(np.array([0.3, -0.2, 1.4, 0.1], dtype=np.float32)), r0)


def test_constant_and_sinusoidal_wind_components():
    """PAPER.md:200, 204 (reading Q40).  CONSTANT: steady air velocity c through the quadratic drag law, evaluated at the start
    of each control step and held -> exact recurrence v <- v + dt (k/m) |c - v| (c - v).  SINUSOIDAL: the printed force of
    episode time, also held over the step."""
    KW, DT = 0.5 * 1.225 * 0.01, 1 / 48
    hov = np.full((1, 4), HOVER, dtype=np.float32)
    res = G - 4 * KF * float(hov[0, 0]) ** 2 / M                     # fp32 hover RPM leaves a tiny vertical residual
    c = np.array([0.9, -0.4, 0.0])
    env, _ = make_env(physics=W.PHYS_MJC, aero_mask=W.AERO_WIND, wind_mask=2, wind_const=list(c), **FREE)
    set_state(env, p=[0, 0, 1.0], q=[1, 0, 0, 0], v=[0, 0, 0], w=[0, 0, 0])
    v = np.zeros(3); p = np.array([0, 0, 1.0])
    for _ in range(96):
        env.step(hov)
        rel = c - v
        a = KW * np.linalg.norm(rel) * rel / M - np.array([0, 0, res])
        p = p + DT * v + 0.5 * DT * DT * a
        v = v + DT * a
    assert np.abs(env.state[0, 7:10] - v).max() < 1e-12 and np.abs(env.state[0, 0:3] - p).max() < 1e-12
    assert 0.2 < v[0] < 0.9 and np.all(env.wind == 0.0)               # drifting downwind, no gust state touched
    # sinusoidal force: v after n steps is the sum of the held accelerations
    A, om = 0.02, 2 * math.pi * 0.7
    env, _ = make_env(physics=W.PHYS_MJC, aero_mask=W.AERO_WIND, wind_mask=8, wind_sine_amp=A, wind_sine_omega=om, **FREE)
    set_state(env, p=[0, 0, 1.0], q=[1, 0, 0, 0], v=[0, 0, 0], w=[0, 0, 0])
    v = np.zeros(3)
    for k in range(60):
        env.step(hov)
        t = k * DT
        v = v + DT * (A * np.array([math.sin(om * t), math.cos(om * t), 0.3 * math.sin(2 * om * t)]) / M - np.array([0, 0, res]))
    assert np.abs(env.state[0, 7:10] - v).max() < 1e-12 and abs(v[1]) > 0.01
    # the components add: DRYDEN + CONSTANT + SINE equals the drag on (gust + c) plus the sine force
    both, _ = make_env(physics=W.PHYS_MJC, aero_mask=W.AERO_WIND, wind_mask=11, wind_const=list(c), wind_sine_amp=A, wind_sine_omega=om, **FREE)
    gust, _ = make_env(physics=W.PHYS_MJC, aero_mask=W.AERO_WIND, wind_mask=1, **FREE)
    for e in (both, gust):
        set_state(e, p=[0, 0, 1.0], q=[1, 0, 0, 0], v=[0, 0, 0], w=[0, 0, 0])
        e.step(hov)
    assert np.array_equal(both.wind, gust.wind)                       # same Philox draw, the gust state excludes c
    u = gust.wind[0] + c
    want = DT * ((KW * np.linalg.norm(u) * u + A * np.array([0.0, 1.0, 0.0])) / M - np.array([0, 0, res]))
    assert np.abs(both.state[0, 7:10] - want).max() < 1e-13


def test_fly_through_waypoint_capture_reward_and_observation():
    """PAPER.md:321 (reading Q41): +10 on capture (distance < 0.1 m), -0.1 |d_wp| shaping, -0.01 |omega| smoothness; the
    default waypoint list; obs = KIN12 + next waypoint + its position in the body frame; the last capture ends the episode."""
    from scipy.spatial.transform import Rotation
    from oracle_util import quat_wxyz_from_scipy
    WPS = np.array([(0, 0, 1), (1, 0, 1), (1, 1, 1.5), (0, 1, 1), (0, 0, 0.5)], dtype=float)
    over = dict(obs_mode=W.OBS_KIN12_WP, reward_mode=W.REW_FLY_THROUGH, target_mode=W.TGT_WAYPOINTS, term_mode=W.TERM_HOVER,
                episode_len_s=20.0, auto_reset=0)
    env, _ = make_env(**over)
    assert np.array_equal(env.targets[0], [0, 0, 1, 0])
    hov = np.full((1, 4), HOVER, dtype=np.float32)
    rot = Rotation.from_euler("ZYX", [0.7, 0.0, 0.0])
    # far from waypoint 0: shaping and smoothness only, target unchanged
    set_state(env, p=[0.5, 0.2, 1.3], q=quat_wxyz_from_scipy(rot), v=[0, 0, 0], w=[0.0, 0.0, 0.3])
    env.step(hov)
    s = env.state[0]
    d = np.linalg.norm(WPS[0] - s[0:3])
    obs, rew, done, _ = env.outputs()
    assert abs(rew[0] - (-0.1 * d - 0.01 * np.linalg.norm(s[10:13]))) < 1e-13 and done[0] == 0
    assert np.array_equal(env.targets[0], [0, 0, 1, 0])
    R = Rotation.from_quat([s[4], s[5], s[6], s[3]])
    assert np.array_equal(obs[0, 12:15], WPS[0]) and np.allclose(obs[0, 15:18], R.inv().apply(WPS[0] - s[0:3]), atol=1e-14)
    # inside the capture radius of waypoint 0: +10 and the chase moves to waypoint 1 (obs already shows it)
    set_state(env, p=[0.03, -0.04, 1.05], q=[1, 0, 0, 0], v=[0, 0, 0], w=[0, 0, 0])
    env.step(hov)
    s = env.state[0]
    d = np.linalg.norm(WPS[0] - s[0:3])
    obs, rew, done, _ = env.outputs()
    assert d < 0.1 and abs(rew[0] - (10.0 - 0.1 * d)) < 1e-9 and done[0] == 0
    assert np.array_equal(env.targets[0], [1, 0, 1, 1]) and np.array_equal(obs[0, 12:15], WPS[1])
    assert np.allclose(obs[0, 15:18], WPS[1] - s[0:3], atol=1e-9)
    # just outside the radius: no capture
    set_state(env, p=[1.0, 0.0, 1.0 + 0.1005], q=[1, 0, 0, 0], v=[0, 0, 0], w=[0, 0, 0])
    env.step(hov)
    assert env.outputs()[1][0] < 0 and np.array_equal(env.targets[0], [1, 0, 1, 1])
    # walk through the rest: the last capture terminates
    for k in range(1, 5):
        set_state(env, p=WPS[k] + [0.01, 0, 0], q=[1, 0, 0, 0], v=[0, 0, 0], w=[0, 0, 0])
        env.step(hov)
        _, rew, done, _ = env.outputs()
        assert rew[0] > 9.9 and done[0] == (1 if k == 4 else 0)
        if k < 4:
            assert np.array_equal(env.targets[0], list(WPS[k + 1]) + [k + 1])


def test_table4_motor_bias_arm_maxrpm_and_initial_state_ranges():
    """Table 4 rows beyond the first eight factors (reading Q39): per-motor thrust bias (4 draws), arm length, MAX_RPM,
    and the "init" row: RPY_0 and v_0 uniform within given half-widths."""
    from scipy.spatial.transform import Rotation
    alpha = [0.0] * 8 + [0.05, 0.02, 0.05, 0.0]
    env, _ = make_env(n_envs=4000, dr_alpha=alpha, reset_rpy_half=[0.1, 0.1, 0.1], reset_vel_half=[0.5, 0.5, 0.5], **FREE)
    f = env.dr
    assert np.all(f[:, :8] == 1.0) and np.all(f[:, 14:] == 1.0)
    assert np.all(np.abs(f[:, 8:12] - 1) <= 0.05) and np.all(np.abs(f[:, 12] - 1) <= 0.02) and np.all(np.abs(f[:, 13] - 1) <= 0.05)
    assert abs(f[:, 8:12].std() - 0.1 / math.sqrt(12)) < 0.002 and np.abs(np.corrcoef(f[:, 8:14].T) - np.eye(6)).max() < 0.06
    st = env.state
    rpy = Rotation.from_quat(st[:, [4, 5, 6, 3]]).as_euler("ZYX")[:, ::-1]           # roll, pitch, yaw
    assert np.abs(rpy).max() <= 0.1 + 1e-12 and np.abs(rpy.std(axis=0) - 0.2 / math.sqrt(12)).max() < 0.003
    assert np.abs(np.linalg.norm(st[:, 3:7], axis=1) - 1).max() < 1e-15
    assert np.abs(st[:, 7:10]).max() <= 0.5 and np.abs(st[:, 7:10].std(axis=0) - 1.0 / math.sqrt(12)).max() < 0.01
    assert np.abs(np.corrcoef(np.hstack([rpy, st[:, 7:10]]).T) - np.eye(6)).max() < 0.06 and np.all(st[:, 10:13] == 0)
    # physics: biases scale each rotor's thrust and reaction torque, the arm scales roll / pitch torque only
    P = O.OracleParams(0)
    env1, _ = make_env(**FREE)
    d = np.ones((1, 16)); d[0, 8:12] = [1.04, 0.97, 1.02, 0.96]; d[0, 12] = 1.015
    env1.dr = d
    set_state(env1, p=[0, 0, 1.0], q=[1, 0, 0, 0], v=[0, 0, 0], w=[0, 0, 0])
    n = float(np.float32(HOVER))
    for _ in range(6):
        env1.step(np.full((1, 4), n, dtype=np.float32))
    F = KF * n * n * d[0, 8:12]
    l = L / math.sqrt(2) * 1.015
    t = 6 / 48
    tx, ty, tz = l * (F[0] + F[1] - F[2] - F[3]), l * (-F[0] + F[1] + F[2] - F[3]), (KM / KF) * (-F[0] + F[1] - F[2] + F[3])
    s = env1.state[0]
    assert abs(s[10] - tx * t / JXX) < 0.03 * abs(s[10]) and abs(s[11] - ty * t / JXX) < 0.1 * abs(s[11])   # gyroscopic coupling aside
    env2, _ = make_env(**FREE)                                  # exact at the first substep: omega = tau h / J
    env2.dr = d
    set_state(env2, p=[0, 0, 1.0], q=[1, 0, 0, 0], v=[0, 0, 0], w=[0, 0, 0])
    Fw, tw = env2.probe_wrench(0, np.full((1, 4), n))
    assert abs(Fw[0, 2] - F.sum()) < 1e-15 and np.allclose(tw[0], [tx, ty, tz], rtol=1e-12, atol=1e-20)
    # MAX_RPM factor < 1 saturates the rotors below the nominal limit; > 1 leaves the nominal command clip in force
    env3, _ = make_env(**FREE)
    d = np.ones((1, 16)); d[0, 13] = 0.96
    env3.dr = d
    set_state(env3, p=[0, 0, 1.0], q=[1, 0, 0, 0], v=[0, 0, 0], w=[0, 0, 0])
    env3.step(np.full((1, 4), 1e6, dtype=np.float32))
    acc = 4 * KF * (0.96 * MAXR) ** 2 / M - G
    assert abs(env3.state[0, 9] - acc / 48) < 1e-10
    d[0, 13] = 1.04
    env3.dr = d
    set_state(env3, p=[0, 0, 1.0], q=[1, 0, 0, 0], v=[0, 0, 0], w=[0, 0, 0])
    env3.step(np.full((1, 4), 1e6, dtype=np.float32))
    assert abs(env3.state[0, 9] - (4 * KF * MAXR ** 2 / M - G) / 48) < 1e-10


def test_per_drone_reward_shares_add_up_and_split_pair_terms():
    """MultiAgentAviary view: each drone's share = its own terms + half of every pair term it is part of."""
    over = dict(reward_mode=W.REW_FORMATION, target_mode=W.TGT_CIRCLE, reset_layout=W.LAYOUT_CIRCLE, circle_radius=0.3, form_radius=0.3,
                form_center=[0, 0, 1], reset_center=[0, 0, 1], **FREE)
    env, _ = make_env(n_envs=1, n_drones=3, **over)
    st = env.state
    st[:, 0:3] = [[0.4, 0.0, 1.0], [-0.1, 0.3, 1.1], [-0.2, -0.2, 0.9]]
    env.state = st
    hov = np.full((3, 4), HOVER, dtype=np.float32)
    env.step(hov)
    p, tg = env.state[:, 0:3], env.targets[:, 0:3]
    want = np.zeros(3)
    for i in range(3):
        want[i] -= np.linalg.norm(p[i] - tg[i])
        for k in range(3):
            if k != i:
                want[i] -= 0.25 * abs(np.linalg.norm(p[i] - p[k]) - np.linalg.norm(tg[i] - tg[k]))
    assert np.allclose(env.reward_per_drone, want, atol=1e-13) and abs(env.reward_per_drone.sum() - env.outputs()[1][0]) < 1e-13
    envh, _ = make_env(n_envs=2, n_drones=2, reward_mode=W.REW_MULTI_HOVER, **FREE)
    envh.step(np.full((4, 4), HOVER, dtype=np.float32))
    assert np.allclose(envh.reward_per_drone.reshape(2, 2).sum(axis=1), envh.outputs()[1], atol=1e-13)


def test_gust_wind_impulses_envelope_and_trigger_rate():
    """PAPER.md:201 (reading Q42): impulses with a sin(pi s) envelope, per-step trigger probability, direction uniform on the
    sphere, speed U(0, gust_max)."""
    KW, DT = 0.5 * 1.225 * 0.01, 1 / 48
    hov = np.full((1, 4), HOVER, dtype=np.float32)
    res = G - 4 * KF * float(hov[0, 0]) ** 2 / M
    # a hand-set impulse: the air velocity follows g sin(pi s) with s = k dt / T, then the impulse ends
    env, _ = make_env(physics=W.PHYS_MJC, aero_mask=W.AERO_WIND, wind_mask=4, gust_prob=0.0, gust_duration=0.25, **FREE)
    set_state(env, p=[0, 0, 1.0], q=[1, 0, 0, 0], v=[0, 0, 0], w=[0, 0, 0])
    g = np.array([0.8, -0.3, 0.2])
    env.gust = np.array([[*g, 0.0]])
    v = np.zeros(3)
    for k in range(20):
        env.step(hov)
        s = k * DT / 0.25
        u = g * math.sin(math.pi * s) if s < 1.0 - 1e-4 else np.zeros(3)      # Q42: over at phase 1 - 1e-4 (12 steps here, not 13)
        rel = u - v
        v = v + DT * (KW * np.linalg.norm(rel) * rel / M - np.array([0, 0, res]))
    assert np.abs(env.state[0, 7:10] - v).max() < 1e-12 and env.gust[0, 3] >= 1.0 - 1e-4 and abs(v[0]) > 1e-3
    # a duration of a whole number of control steps lasts exactly that many: the phase stops advancing after the 12th
    assert abs(env.gust[0, 3] - 1.0) < 1e-12
    # trigger statistics over many envs: fraction of envs whose impulse started in the first step = gust_prob;
    # speeds uniform in [0, gust_max]; directions isotropic
    N = 20000
    env, _ = make_env(n_envs=N, physics=W.PHYS_MJC, aero_mask=W.AERO_WIND, wind_mask=4, gust_prob=0.1, gust_max=2.0, gust_duration=10.0, **FREE)
    env.step(np.tile(hov, (N, 1)))
    gs = env.gust
    on = gs[:, 3] < 1.0
    assert abs(on.mean() - 0.1) < 0.01 and np.all(gs[~on, :3] == 0.0)
    sp = np.linalg.norm(gs[on, :3], axis=1)
    assert sp.max() <= 2.0 and abs(sp.mean() - 1.0) < 0.05 and abs(sp.std() - 2 / math.sqrt(12)) < 0.05
    d = gs[on, :3] / sp[:, None]
    assert np.abs(d.mean(axis=0)).max() < 0.05 and np.abs((d ** 2).mean(axis=0) - 1 / 3).max() < 0.03
    assert np.allclose(gs[on, 3], DT / 10.0)                          # progress after the first sample


def test_kin12_z_observation_is_state_plus_target_altitude():
    """PAPER.md:317 / 333: MultiHoverAviary and MultiAgentAviary observe 13 numbers per drone: KIN12 + its target altitude."""
    env, _ = make_env(n_envs=3, n_drones=4, obs_mode=W.OBS_KIN12_Z, reward_mode=W.REW_MULTI_HOVER, target_mode=W.TGT_SPAWN_LINSPACE,
                      mh_z_lo=0.7, mh_z_hi=1.2, **FREE)
    obs = env.outputs()[0].reshape(3, 4, 13)
    assert np.allclose(obs[:, :, 12], np.linspace(0.7, 1.2, 4)[None, :], atol=1e-15)
    st = env.state.reshape(3, 4, 13)
    assert np.array_equal(obs[:, :, 0:3], st[:, :, 0:3]) and np.array_equal(obs[:, :, 6:9], st[:, :, 7:10]) and np.array_equal(obs[:, :, 9:12], st[:, :, 10:13])


def test_race_parameters_of_the_waypoint_task_family():
    """RaceAviary (reading Q43): +20 per gate, +2 |v| speed bonus, -0.05 d_gate shaping, the track run twice."""
    gates = [1.5, 0.0, 1.0, 0.75, 1.3, 1.0, -0.75, 1.3, 1.0, -1.5, 0.0, 1.0, -0.75, -1.3, 1.0, 0.75, -1.3, 1.0]
    env, _ = make_env(obs_mode=W.OBS_KIN12_WP, reward_mode=W.REW_FLY_THROUGH, target_mode=W.TGT_WAYPOINTS, n_waypoints=6,
                      waypoints=gates + [0.0] * 6, wp_radius=0.2, wp_bonus=20.0, wp_shaping=0.05, wp_speed=2.0, wp_omega=0.0, wp_laps=2,
                      term_mode=W.TERM_HOVER, episode_len_s=30.0, auto_reset=0)
    hov = np.full((1, 4), HOVER, dtype=np.float32)
    G6 = np.array(gates).reshape(6, 3)
    set_state(env, p=[1.0, 0.0, 1.0], q=[1, 0, 0, 0], v=[0.6, 0.8, 0.0], w=[0.0, 0.0, 1.0])
    env.step(hov)
    s = env.state[0]
    want = 2.0 * np.linalg.norm(s[7:10]) - 0.05 * np.linalg.norm(G6[0] - s[0:3])
    assert abs(env.outputs()[1][0] - want) < 1e-12 and abs(np.linalg.norm(s[7:10]) - 1.0) < 1e-6
    idx = 0
    for lap in range(2):
        for k in range(6):
            set_state(env, p=G6[k] + [0.0, 0.05, 0.0], q=[1, 0, 0, 0], v=[0, 0, 0], w=[0, 0, 0])
            env.step(hov)
            _, rew, done, _ = env.outputs()
            idx += 1
            assert abs(rew[0] - (20.0 - 0.05 * 0.05)) < 1e-6 and done[0] == (1 if idx == 12 else 0)
            if idx < 12:
                assert np.allclose(env.targets[0], list(G6[idx % 6]) + [idx])


def test_motor_lag_first_order_rotor_dynamics():
    """Table 4 "motor lag tau_mot U[5, 50] ms (per ep.)", reading Q44: rotor speeds follow the command through a first-order
    lag sampled exactly per substep, n <- n + (1 - e^(-h/tau)) (n_cmd - n); episodes start at hover speed."""
    h = 1 / 240
    env, _ = make_env(n_envs=3000, motor_lag_lo=0.005, motor_lag_hi=0.05, **FREE)
    tau = env.dr[:, 14]
    assert tau.min() >= 0.005 and tau.max() <= 0.05 and abs(tau.mean() - 0.0275) < 0.001 and abs(tau.std() - 0.045 / math.sqrt(12)) < 0.0007
    assert np.allclose(env.rotor, HOVER, rtol=1e-15) and np.all(env.dr[:, :14] == 1.0)
    # one drone, tau fixed by hand: a thrust step from hover
    env, _ = make_env(motor_lag_lo=0.02, motor_lag_hi=0.02, **FREE)
    assert abs(env.dr[0, 14] - 0.02) < 1e-15
    set_state(env, p=[0, 0, 1.0], q=[1, 0, 0, 0], v=[0, 0, 0], w=[0, 0, 0])
    n1 = float(np.float32(1.2 * HOVER))
    a = np.full((1, 4), n1, dtype=np.float32)
    n, v, z = HOVER, 0.0, 1.0
    gam = 1 - math.exp(-h / 0.02)
    for step in range(12):
        env.step(a)
        for k in range(5):
            n = n + gam * (n1 - n)
            acc = 4 * KF * n * n / M - G
            z = z + h * v + 0.5 * h * h * acc
            v = v + h * acc
    assert abs(env.state[0, 9] - v) < 1e-12 and abs(env.state[0, 2] - z) < 1e-12 and np.allclose(env.rotor[0], n, rtol=1e-14)
    assert abs(n - (n1 + (HOVER - n1) * math.exp(-60 * h / 0.02))) < 1e-9 * n1       # the closed form of the lag itself
    # the lag applies rotor by rotor: a differential command builds torque gradually (smaller rate than without lag)
    env2, _ = make_env(**FREE)
    for e in (env, env2):
        set_state(e, p=[0, 0, 1.0], q=[1, 0, 0, 0], v=[0, 0, 0], w=[0, 0, 0])
    env.rotor = np.full((1, 4), HOVER)
    b = (np.array([[1.05, 1.05, 0.95, 0.95]]) * HOVER).astype(np.float32)
    env.step(b); env2.step(b)
    assert 0 < env.state[0, 10] < 0.6 * env2.state[0, 10]
