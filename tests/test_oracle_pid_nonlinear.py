"""Pins of the cascaded PID outside its linear regime (Eq.9, T = m |a*|, the small-angle attitude target, the
clamped allocation inverse) on hand-built states: yawed vehicles, waypoints far along each world axis, saturated tilt targets,
torque clamps and a saturated mixer.  Expected values are evaluated here from the printed formulas with Table 6's gains
(K_p = (0.4, 0.4, 1.0), K_i = 0.01, attitude K_p = (2e-3, 2e-3, 1e-3), K_i = (0, 0, 1e-4), K_d = (5e-4, 5e-4, 2e-4)),
never by the oracle.  A cos psi / sin psi swap, a wrong sign in the tilt map, |a*| replaced by a*_z, or a clamp applied to
the wrong quantity fails one of them.  Also here: the Box-Muller word -> component map of the wind draw, pinned through the
simulator's own first gust update and computed in numpy from the raw Philox words.
"""
import math

import numpy as np
import pytest

from oracle import oracle as O
from oracle_util import FREE, make_env, set_state
from paper_2606_08039_b200 import workloads as W

M, G, DT = 0.027, 9.81, 1.0 / 48.0
KF = 3.16e-10
L_ARM = 0.0397 / math.sqrt(2.0)
KAPPA = 7.94e-12 / 3.16e-10


def yawed(psi):
    return [math.cos(psi / 2), 0.0, 0.0, math.sin(psi / 2)]


def decode(env, P, action):
    rpm = env.probe_decode(np.array(action, dtype=np.float32))
    T, tau, _ = O.motor_wrench(P, rpm[0])
    return rpm[0], T, tau


@pytest.mark.parametrize("psi", [0.75, -2.125])        # exactly representable in the fp32 action row
@pytest.mark.parametrize("axis,sign", [(0, +1), (0, -1), (1, +1), (1, -1)])
def test_lateral_waypoint_under_yaw_unsaturated_and_saturated(psi, axis, sign):
    for d, saturated in ((5.0, False), (30.0, True)):
        env, P = make_env(action=W.ACT_PID, **FREE)
        set_state(env, p=[0, 0, 1.0], q=yawed(psi), v=[0, 0, 0], w=[0, 0, 0])
        wp = [0.0, 0.0, 1.0, psi]
        wp[axis] = sign * d
        _, T, tau = decode(env, P, wp)
        e = sign * d
        a_lat = 0.4 * e + 0.01 * (e * DT)                       # Eq.9: K_p e + K_i I, I = e dt after the first update
        ax, ay = (a_lat, 0.0) if axis == 0 else (0.0, a_lat)
        phi = (ax * math.sin(psi) - ay * math.cos(psi)) / G      # the printed small-angle map
        th = (ax * math.cos(psi) + ay * math.sin(psi)) / G
        if saturated:
            assert abs(phi) > 0.5 and abs(th) > 0.5              # the case really saturates both
        phi_c, th_c = max(-0.5, min(0.5, phi)), max(-0.5, min(0.5, th))
        assert abs(T - M * math.sqrt(a_lat ** 2 + G ** 2)) < 1e-12               # T = m |a*|, not m a*_z
        assert abs(tau[0] - 2e-3 * phi_c) < 1e-12 and abs(tau[1] - 2e-3 * th_c) < 1e-12 and abs(tau[2]) < 1e-12
        assert (tau[0] > 0) == (phi > 0) and (tau[1] > 0) == (th > 0)


def test_hand_values_of_one_yawed_case():
    """psi = 0.75, waypoint 5 m along +x: the numbers themselves, worked out by hand."""
    env, P = make_env(action=W.ACT_PID, **FREE)
    set_state(env, p=[0, 0, 1.0], q=yawed(0.75), v=[0, 0, 0], w=[0, 0, 0])
    _, T, tau = decode(env, P, [5.0, 0.0, 1.0, 0.75])
    # a*_x = 0.4 * 5 + 0.01 * 5/48 = 2.001041667; phi* = a*_x sin 0.75 / 9.81 = 0.13904053; theta* = a*_x cos 0.75 / 9.81 = 0.14924974
    assert abs(tau[0] - 2.7808105e-4) < 2e-11 and abs(tau[1] - 2.9849947e-4) < 2e-11
    assert abs(T - 0.27032417) < 1e-8                                              # 0.027 * sqrt(2.001041667^2 + 9.81^2)


def test_vertical_waypoint_keeps_level_and_saturates_thrust():
    for psi in (0.75, -2.125):
        env, P = make_env(action=W.ACT_PID, **FREE)
        set_state(env, p=[0, 0, 1.0], q=yawed(psi), v=[0, 0, 0], w=[0, 0, 0])
        rpm, T, tau = decode(env, P, [0.0, 0.0, 501.0, psi])
        assert np.allclose(rpm, P.derived()["max_rpm"], rtol=1e-12) and np.abs(tau).max() < 1e-12
        rpm, T, tau = decode(env, P, [0.0, 0.0, 1.5, psi])
        assert abs(T - M * (1.0 * 0.5 + 0.01 * 0.5 * DT + G)) < 1e-12 and np.abs(tau).max() < 1e-12


def test_velocity_error_and_feed_forward_enter_eq9():
    env, P = make_env(action=W.ACT_PID, a_ff=[0.3, -0.2, 0.1], **FREE)
    set_state(env, p=[0, 0, 1.0], q=yawed(0.0), v=[0.5, -0.25, 0.125], w=[0, 0, 0])
    _, T, tau = decode(env, P, [0.0, 0.0, 1.0, 0.0])
    ax, ay, az = 0.9 * (-0.5) + 0.3, 0.9 * 0.25 - 0.2, 2.0 * (-0.125) + 0.1 + G      # K_d (v* - v) + a_ff + g z
    assert abs(T - M * math.sqrt(ax * ax + ay * ay + az * az)) < 1e-12
    assert abs(tau[0] - 2e-3 * (-ay / G)) < 1e-12 and abs(tau[1] - 2e-3 * (ax / G)) < 1e-12


def test_torque_clamps_under_yaw_and_the_saturated_mixer():
    """Body rates and a yaw error large enough for all three torque clamps, with a waypoint far BELOW so that the thrust is
    small and the per-rotor clip to [0, s_max] bites: the rotor speeds themselves against the hand-evaluated mixer."""
    psi = 0.75
    env, P = make_env(action=W.ACT_PID, **FREE)
    set_state(env, p=[0, 0, 9.0], q=yawed(psi), v=[0, 0, 0], w=[10.0, -10.0, 0.0])
    rpm, _, _ = decode(env, P, [0.0, 0.0, 1.0, psi + 3.0])
    txy, tz = P.get("tau_xy_max"), P.get("tau_z_max")
    assert abs(txy - 4 * L_ARM * (M * G / 4) / 3) < 1e-9 and abs(tz - 4 * KAPPA * (M * G / 4) / 3) < 1e-9      # reading Q17 (float32 defaults)
    az = 1.0 * (-8.0) + 0.01 * (-8.0 * DT) + G
    T = M * abs(az)
    tau = [-txy, +txy, +tz]            # -K_d w_x = -5e-3 -> -clamp; -K_d w_y = +5e-3 -> +clamp; K_p 3 + K_i 3/48 = 3.00625e-3 -> +clamp
    a, b, c = tau[0] / L_ARM, tau[1] / L_ARM, tau[2] / KAPPA
    s = [0.25 * (T + a - b - c), 0.25 * (T + a + b + c), 0.25 * (T - a + b - c), 0.25 * (T - a - b + c)]
    s_max = KF * P.derived()["max_rpm"] ** 2
    expect = [math.sqrt(min(max(x, 0.0), s_max) / KF) for x in s]
    assert min(s) < 0 < max(s)                                                         # the clip really acts
    assert np.allclose(rpm, expect, rtol=1e-9, atol=1e-6)


def test_vel_action_rotates_the_command_by_the_heading_only():
    """Reading Q20 under a tilted attitude: the command frame is the yaw-only heading frame, whatever roll and pitch are."""
    from scipy.spatial.transform import Rotation
    psi = -2.1
    r = Rotation.from_euler("ZYX", [psi, 0.2, -0.15])
    x, y, z, w = r.as_quat()
    env, P = make_env(action=W.ACT_VEL, **FREE)
    set_state(env, p=[0, 0, 1.0], q=[w, x, y, z], v=[0, 0, 0], w=[0, 0, 0])
    _, T, tau = decode(env, P, [0.5, 0.0, 0.0, 0.0])
    vx, vy = 0.5 * math.cos(psi), 0.5 * math.sin(psi)
    ax, ay = 0.9 * vx, 0.9 * vy
    assert abs(T - M * math.sqrt(ax * ax + ay * ay + G * G)) < 1e-9
    phi_ref = (ax * math.sin(psi) - ay * math.cos(psi)) / G          # = 0: a command along the heading asks for pitch only
    th_ref = (ax * math.cos(psi) + ay * math.sin(psi)) / G
    assert abs(phi_ref) < 1e-12 and abs(th_ref - 0.9 * 0.5 / G) < 1e-12
    assert abs(tau[0] - 2e-3 * (phi_ref - (-0.15))) < 1e-9 and abs(tau[1] - 2e-3 * (th_ref - 0.2)) < 1e-9


def test_box_muller_word_to_component_map_through_the_first_gust_update():
    """O12 / PAPER.md:203: words (0, 1) -> xi_0 = r cos, xi_1 = r sin; words (2, 3) -> xi_2 = r' cos.  From a calm start the first
    AR(1) update leaves w = sigma sqrt(1 - alpha^2) xi, so the simulator's own wind state exposes xi; the expected values come from
    the raw Philox words (counter = env, 0xFFFFFFFF, t = 1, stream 2) through numpy."""
    seed, N = (9 << 32) | 1234, 64
    P = O.OracleParams(0, aero_mask=W.AERO_WIND, wind_sigma=0.5, wind_tau=1.0, k_wind=0.0, **FREE)
    env = O.OracleEnv(N, 1, W.PHYS_MJC, W.ACT_RPM, P)
    env.reset(seed)
    env.step(np.full((N, 4), 14000.0, dtype=np.float32))
    alpha = math.exp(-DT / 1.0)
    gain = 0.5 * math.sqrt(1.0 - alpha * alpha)
    for e in range(N):
        x = O.philox([e, 0xFFFFFFFF, 1, 2], [1234, 9]).astype(np.uint64)
        u = (x >> np.uint64(8)).astype(np.float64) / 2.0 ** 24
        r1, r2 = math.sqrt(-2.0 * math.log(1.0 - u[0])), math.sqrt(-2.0 * math.log(1.0 - u[2]))
        xi = np.array([r1 * math.cos(2 * math.pi * u[1]), r1 * math.sin(2 * math.pi * u[1]), r2 * math.cos(2 * math.pi * u[3])])
        assert np.abs(env.wind[e] - gain * xi).max() < 1e-13, e
