"""Pins of the oracle's sensor rows of Table 4 (position / vel / RPY noise N(0, 1 cm / 5 cm/s / 1 deg),
gyro noise N(0, 0.05 rad/s), per step) and the sticky per-episode observation bias of PAPER.md:248 (iii); reading Q49.
Expected values are the table's standard deviations, the defining properties of independent zero-mean Gaussian noise
(checked with scipy's distribution tests) and structural facts (which columns move, what stays fixed over an episode);
none comes from the oracle or the CUDA path."""
import math

import numpy as np
from scipy import stats

from oracle_util import FREE, make_env
from paper_2606_08039_b200 import workloads as W

TABLE4 = [0.01, 0.05, math.radians(1.0), 0.05]          # position m, velocity m/s, RPY rad, gyro rad/s
GROUP_COLS = {0: [0, 1, 2], 1: [6, 7, 8], 2: [3, 4, 5], 3: [9, 10, 11]}      # KIN12 row = [p, eta, v, omega]
HOVER = W.hover_rpm_f32()
SPREAD = dict(reset_center=[0, 0, 1], reset_half=[0.1, 0.1, 0.1], reset_rpy_half=[0.1, 0.1, 0.1], reset_vel_half=[0.5, 0.5, 0.5])


def run(n_envs, steps, n_drones=1, seed=7, **over):
    """Hover-RPM rollout; returns the observation after every step (and after the reset), the state and done flags."""
    env, _ = make_env(n_envs=n_envs, n_drones=n_drones, **over)
    env.reset(seed)
    act = np.full((n_envs * n_drones, 4), HOVER, dtype=np.float32)
    obs, dones = [env.outputs()[0].copy()], []
    for _ in range(steps):
        env.step(act)
        o, _, d, _ = env.outputs()
        obs.append(o.copy()); dones.append(d.copy())
    return env, np.array(obs), np.array(dones)


def test_noise_has_the_table4_standard_deviations_is_gaussian_and_leaves_the_state_alone():
    N = 20000
    env0, clean, _ = run(N, 3, **SPREAD, **FREE)
    env1, noisy, _ = run(N, 3, obs_noise=TABLE4, **SPREAD, **FREE)
    assert np.array_equal(env0.state, env1.state)                      # only the emitted observation is perturbed
    res = noisy - clean                                                # [steps + 1, N, 12]
    assert np.abs(clean[0]).max() > 0.05                               # the clean rows are not trivially zero
    for k in range(res.shape[0]):                                      # the reset's observation is noisy too
        for g, cols in GROUP_COLS.items():
            for c in cols:
                x = res[k, :, c]
                assert abs(x.std() / TABLE4[g] - 1.0) < 0.03, (k, c, x.std())          # std error of the std: 0.5 %
                assert abs(x.mean()) < 5 * TABLE4[g] / math.sqrt(N), (k, c, x.mean())
                assert stats.kstest(x / TABLE4[g], "norm").pvalue > 1e-3, (k, c)
    # independence: across the 12 entries of a row, and across consecutive steps (fresh draws every step)
    z = res[1] / res[1].std(axis=0)
    cc = np.corrcoef(z.T)
    assert np.abs(cc - np.eye(12)).max() < 5 / math.sqrt(N)
    for c in range(12):
        assert abs(np.corrcoef(res[1, :, c], res[2, :, c])[0, 1]) < 5 / math.sqrt(N)
    # the two Box-Muller outputs of one uniform pair are uncorrelated but share a radius: x^2 + y^2 is chi^2 with 2 dof
    r2 = (res[1, :, 0] / TABLE4[0]) ** 2 + (res[1, :, 1] / TABLE4[0]) ** 2
    assert stats.kstest(r2, "chi2", args=(2,)).pvalue > 1e-3


def test_each_sigma_moves_only_its_own_columns_in_every_observation_layout():
    N = 64
    layouts = {
        W.OBS_KIN12: ({0: [0, 1, 2], 1: [6, 7, 8], 2: [3, 4, 5], 3: [9, 10, 11]}, 12, 1, {}),
        W.OBS_KIN20: ({0: [0, 1, 2], 1: [10, 11, 12], 2: [7, 8, 9], 3: [13, 14, 15]}, 20, 1, {}),       # [p, q, eta, v, omega, a]
        W.OBS_KIN12_TGT: ({0: [0, 1, 2], 1: [6, 7, 8], 2: [3, 4, 5], 3: [9, 10, 11]}, 16, 1,
                          dict(target_mode=W.TGT_BOX, target_lo=[-1, -1, 0.5], target_hi=[1, 1, 1.5])),
        W.OBS_KIN12_ADJ: ({0: [0, 1, 2], 1: [6, 7, 8], 2: [3, 4, 5], 3: [9, 10, 11]}, 15, 3, dict(adj_radius=0.5, reset_layout=W.LAYOUT_CIRCLE, circle_radius=0.3)),
    }
    for mode, (groups, opd, M, extra) in layouts.items():
        base = dict(obs_mode=mode, **extra, **SPREAD, **FREE)
        _, clean, _ = run(N, 2, n_drones=M, **base)
        assert clean.shape[2] == opd * M
        for g, cols in groups.items():
            for field in ("obs_noise", "obs_bias"):
                sig = [0.0] * 4
                sig[g] = 0.25
                _, noisy, _ = run(N, 2, n_drones=M, **{field: sig}, **base)
                moved = (np.abs(noisy - clean) > 0).any(axis=(0, 1)).reshape(M, opd)
                want = np.zeros(opd, dtype=bool)
                want[cols] = True
                assert (moved == want).all(), (mode, g, field, moved)


def test_bias_is_fixed_over_an_episode_redrawn_at_the_auto_reset_and_adds_in_quadrature():
    N, steps = 6000, 12
    ep = dict(term_mode=W.TERM_NONE, auto_reset=1, episode_len_s=5.0 / 48.0)               # truncation after 5 control steps
    _, clean, dones = run(N, steps, **SPREAD, **ep)
    _, biased, dones_b = run(N, steps, obs_bias=TABLE4, **SPREAD, **ep)
    assert np.array_equal(dones, dones_b) and (dones[4] == 2).all() and (dones[9] == 2).all() and dones[:4].max() == 0
    res = biased - clean                                               # index k: the observation after step k (0 = reset)
    # episode 1 = observations 0..4, episode 2 = 5..9 (the auto-reset of step 5 opens it), episode 3 = 10..
    for a, b in [(0, 4), (5, 9), (10, 12)]:
        for k in range(a, b + 1):
            assert np.abs(res[k] - res[a]).max() < 1e-12, k           # same additive term all episode long
    for g, cols in GROUP_COLS.items():
        for c in cols:
            for k in (0, 5, 10):
                assert abs(res[k, :, c].std() / TABLE4[g] - 1.0) < 0.05
                assert stats.kstest(res[k, :, c] / TABLE4[g], "norm").pvalue > 1e-3
            assert abs(np.corrcoef(res[0, :, c], res[5, :, c])[0, 1]) < 5 / math.sqrt(N)   # a new draw per episode
            assert abs(np.corrcoef(res[5, :, c], res[10, :, c])[0, 1]) < 5 / math.sqrt(N)
    # noise and bias together: independent terms, variances add
    _, both, _ = run(N, 2, obs_noise=TABLE4, obs_bias=[3 * s for s in TABLE4], **SPREAD, **FREE)
    _, clean2, _ = run(N, 2, **SPREAD, **FREE)
    r = both - clean2
    for g, cols in GROUP_COLS.items():
        for c in cols:
            assert abs(r[1, :, c].std() / (TABLE4[g] * math.sqrt(10.0)) - 1.0) < 0.05
            assert abs(np.corrcoef(r[1, :, c], r[2, :, c])[0, 1] - 0.9) < 0.02     # shared bias: corr = 9 / (9 + 1)


def test_noise_is_keyed_by_global_env_drone_and_step():
    base = dict(obs_noise=TABLE4, obs_bias=TABLE4, **SPREAD, **FREE)
    _, whole, _ = run(12, 3, n_drones=2, **base)
    _, part, _ = run(4, 3, n_drones=2, env_index_base=5, **base)       # envs 5..8 of the unsplit batch
    assert np.array_equal(whole[:, 5:9], part)
    _, other, _ = run(12, 3, n_drones=2, seed=8, **base)
    assert np.abs(whole - other).min() > 0                             # another seed: every entry differs
    # the two drones of an env and two envs draw different values
    assert np.abs(whole[1, :, :12] - whole[1, :, 12:]).min() > 0 and np.abs(whole[1, 0] - whole[1, 1]).min() > 0
