"""Pins of the oracle's altitude-dependent Dryden gust ("L_u = h/(0.177 + 8.23e-4 h)^1.2 at altitude h. The
discrete-time recursion is x <- alpha x + sigma sqrt(1 - alpha^2) xi with alpha = e^(-dt V / L)"; reading Q50).  Expected values
are the printed formulas evaluated here at hand-picked altitudes, the AR(1) statistics they imply, and the fixed-tau form as
the V = 0 special case."""
import math

import numpy as np

from oracle import oracle as O
from oracle_util import FREE, make_env, set_state
from paper_2606_08039_b200 import workloads as W

DT = 1.0 / 48.0
HOVER = W.hover_rpm_f32()


def L_u(h):
    return h / (0.177 + 8.23e-4 * h) ** 1.2


def test_printed_length_scale_values():
    # hand arithmetic: (0.177823)^1.2 = exp(1.2 ln 0.177823) = exp(-2.072365) = 0.125888 -> L_u(1 m) = 7.9436 m
    assert abs(L_u(1.0) - 7.9436) < 2e-3
    assert abs(L_u(0.3) - 0.3 / 0.125363) < 2e-3            # (0.1772469)^1.2 = 0.125363


def test_first_update_uses_alpha_of_the_env_mean_altitude():
    V, sigma = 6.0, 0.5
    for heights in ([1.0], [0.3], [2.5], [0.5, 1.5], [0.2, 0.4, 2.4]):
        M = len(heights)
        env, _ = make_env(n_drones=M, aero_mask=W.AERO_WIND, dryden_airspeed=V, k_wind=0.0, **FREE)
        env.reset(42)
        s = env.state
        s[:, 0:3] = [[0.7 * i, 0.0, h] for i, h in enumerate(heights)]
        env.state = s
        act = np.full((M, 4), HOVER, dtype=np.float32)
        env.step(act)
        alpha = math.exp(-DT * V / L_u(sum(heights) / M))
        xi1 = O.wind_normals(42, 0, 1)
        assert np.allclose(env.wind[0], sigma * math.sqrt(1 - alpha ** 2) * xi1, rtol=1e-12), heights
        w1 = env.wind[0].copy()
        env.step(act)                                                   # k_wind = 0 at hover thrust: the altitude has not moved
        assert np.allclose(env.wind[0], alpha * w1 + sigma * math.sqrt(1 - alpha ** 2) * O.wind_normals(42, 0, 2), rtol=1e-9)
    # below dryden_h_min the floor value is used (default 0.05 m); V = 0 is the fixed-tau recursion of Q27
    env, _ = make_env(aero_mask=W.AERO_WIND, dryden_airspeed=V, k_wind=0.0, **FREE)
    env.reset(42)
    set_state(env, p=[0, 0, 0.01], q=[1, 0, 0, 0], v=[0, 0, 0], w=[0, 0, 0])
    env.step(np.full((1, 4), HOVER, dtype=np.float32))
    alpha = math.exp(-DT * V / L_u(0.05))
    assert np.allclose(env.wind[0], sigma * math.sqrt(1 - alpha ** 2) * O.wind_normals(42, 0, 1), rtol=1e-12)
    env, _ = make_env(aero_mask=W.AERO_WIND, dryden_airspeed=0.0, **FREE)
    env.reset(42)
    env.step(np.zeros((1, 4), dtype=np.float32))
    alpha = math.exp(-DT / 1.0)
    assert np.allclose(env.wind[0], sigma * math.sqrt(1 - alpha ** 2) * O.wind_normals(42, 0, 1), rtol=1e-12)


def test_stationary_statistics_follow_the_altitude():
    """Hovering at fixed altitude (no wind force: k_wind = 0) the gust is AR(1) with lag-1 correlation alpha(h) and variance
    sigma^2: low flight decorrelates faster (smaller L_u)."""
    N, V = 3000, 8.0
    seen = {}
    for h in (0.3, 1.0, 2.5):
        env, _ = make_env(n_envs=N, aero_mask=W.AERO_WIND, dryden_airspeed=V, k_wind=0.0, wind_sigma=0.7, threads=8,
                          reset_center=[0, 0, h], reset_half=[0, 0, 0], **FREE)
        env.reset(5)
        act = np.full((N, 4), HOVER, dtype=np.float32)
        hist = []
        for t in range(420):
            env.step(act)
            if t >= 300:
                hist.append(env.wind.copy())
        assert np.abs(env.state[:, 2] - h).max() < 1e-4                  # fp32-rounded hover RPM: a few micrometres of drift
        hist = np.array(hist)
        alpha = math.exp(-DT * V / L_u(h))
        c1 = (hist[1:] * hist[:-1]).mean(axis=(0, 1)) / (hist * hist).mean(axis=(0, 1))
        assert np.abs(c1 - alpha).max() < 0.01, (h, c1, alpha)
        assert np.abs(hist.var(axis=(0, 1)) / 0.49 - 1).max() < 0.05, h
        seen[h] = c1.mean()
    assert seen[0.3] < seen[1.0] < seen[2.5]
