"""CUDA path vs float64 oracle, element by element on the same seeded inputs (BASELINE.json criteria).

Tolerances (north_star): after 1 s of simulated time |dp| <= 1e-4 m, |dv| <= 1e-3 m/s, |dq| <= 1e-4
(sign-aligned), reward <= 1e-3 relative, done / reset indices bit-exact.  Where fp32 and fp64 can
legitimately take different sides of a threshold (the oracle reports its distance to the nearest
threshold per env and step), a mismatch with margin < 1e-4 is a "tie": that env is dropped from the
rest of the comparison and counted; a mismatch with a larger margin is a failure.

Conditioning.  Eq.6's downwash is violently unstable when one drone passes closely under another
(several N on a 0.26 N vehicle, stiffness ~1e3 s^-2: errors double every control step), so for such an
env no fp32 computation can stay within 1e-4 m of the fp64 one for a second.  To separate that from a
formula error, a SHADOW oracle runs beside the reference one on the same actions with its state rounded
to fp32 after every control step (the smallest perturbation any fp32 implementation must make).  An
env whose shadow drifts from the reference by more than tolerance/20 (SURVEY.md §8(c) measured a >=20x
margin for a faithful fp32 path) is "ill-conditioned": it is dropped from the comparison and counted,
and the count is bounded per config.  Every other env must meet the tolerances above.
"""
import os

import numpy as np

from oracle import oracle as O
from paper_2606_08039_b200 import workloads as W

TOL_P, TOL_V, TOL_Q, TOL_W, TOL_R, TIE = 1e-4, 1e-3, 1e-4, 1e-3, 1e-3, 1e-4
R_FLOOR = 1e-5      # absolute floor of the reward comparison: |dr| <= TOL_R |r| + R_FLOOR (rewards pass through zero; fp32 rounding of a sum of O(1) terms)


def reward_err(r32, r64):
    """Reward error in units of its tolerance (<= 1 passes): north_star's 1e-3 RELATIVE error, with the stated absolute floor."""
    return np.abs(r32 - r64) / (TOL_R * np.abs(r64) + R_FLOOR)


def make_pair(wl, extra=None, model=0):
    import paper_2606_08039_b200 as mdg
    over = dict(wl.params)
    if extra:
        over.update(extra)
    orc = O.OracleEnv(wl.n_envs, wl.n_drones, wl.physics_mode, wl.action_type, O.OracleParams(model, **over),
                      n_threads=os.cpu_count() or 1)
    gpu = mdg.Env(wl.n_envs, wl.n_drones, wl.physics_mode, wl.action_type, mdg.default_params(model, **over))
    return orc, gpu


def actions_for(wl, orc, gpu, t):
    """Same fp32 action array for both sides; the two Philox implementations are first checked bit-equal."""
    import torch
    kind = wl.actions[0]
    if kind == "targets":
        a = orc.targets.astype(np.float32)
        return a, torch.from_numpy(a).cuda()
    base = W.hover_rpm_f32() if kind == "hover_scale" else 1.0
    a = O.gen_actions(wl.seed, t, wl.n_envs, wl.n_drones, base, wl.actions[1], wl.actions[2])
    a_dev = gpu.gen_actions(wl.seed, t, base, wl.actions[1], wl.actions[2])
    assert np.array_equal(a_dev.cpu().numpy(), a), "host and device Philox action streams differ"
    return a, a_dev


def compare_state(orc, gpu, alive_env, M, label):
    s64 = orc.state
    g = gpu.get_state()
    s32 = g["state"].astype(np.float64)
    alive = np.repeat(alive_env, M)
    dp = np.abs(s32[:, 0:3] - s64[:, 0:3]).max(axis=1)
    dv = np.abs(s32[:, 7:10] - s64[:, 7:10]).max(axis=1)
    dw = np.abs(s32[:, 10:13] - s64[:, 10:13]).max(axis=1)
    dq = np.minimum(np.abs(s32[:, 3:7] - s64[:, 3:7]).max(axis=1), np.abs(s32[:, 3:7] + s64[:, 3:7]).max(axis=1))
    res = dict(dp=dp[alive].max(initial=0), dv=dv[alive].max(initial=0), dq=dq[alive].max(initial=0), dw=dw[alive].max(initial=0))
    assert res["dp"] <= TOL_P and res["dv"] <= TOL_V and res["dq"] <= TOL_Q and res["dw"] <= TOL_W, (label, res)
    return res, g


def shadow_drift(orc, shadow, M):
    """Per-env flag: the fp32-rounded shadow left the reference oracle by more than tolerance/20."""
    a, b = orc.state, shadow.state
    dp = np.abs(a[:, 0:3] - b[:, 0:3]).max(axis=1)
    dv = np.abs(a[:, 7:10] - b[:, 7:10]).max(axis=1)
    dq = np.minimum(np.abs(a[:, 3:7] - b[:, 3:7]).max(axis=1), np.abs(a[:, 3:7] + b[:, 3:7]).max(axis=1))
    bad = (dp > TOL_P / 20) | (dv > TOL_V / 20) | (dq > TOL_Q / 20)
    bad = bad.reshape(-1, M).any(axis=1)
    bad |= orc.outputs()[2] != shadow.outputs()[2]
    bad |= orc.ep_step != shadow.ep_step
    return bad


def run_parity(wl, steps=48, extra=None, check_every=8, max_ill_frac=0.0, model=0):
    orc, gpu = make_pair(wl, extra, model)
    over = dict(wl.params)
    over.update(extra or {})
    shadow = O.OracleEnv(wl.n_envs, wl.n_drones, wl.physics_mode, wl.action_type, O.OracleParams(model, **over),
                         n_threads=os.cpu_count() or 1)
    N, M = wl.n_envs, wl.n_drones
    orc.reset(wl.seed)
    shadow.reset(wl.seed)
    gpu.reset(wl.seed)
    alive = np.ones(N, dtype=bool)
    ill = np.zeros(N, dtype=bool)
    res0, g = compare_state(orc, gpu, alive, M, "reset")
    assert res0["dp"] < 1e-6
    assert np.abs(g["targets"] - orc.targets).max() < 1e-6
    o64 = orc.outputs()[0]
    assert np.abs(gpu.obs.cpu().numpy() - o64).max() < 1e-6
    opd = gpu.obs_dim // M
    ties = dict(done=0, reward=0, adj=0)
    worst = dict(dp=0.0, dv=0.0, dq=0.0, dw=0.0, rew=0.0)
    n_done = 0
    for t in range(steps):
        a, a_dev = actions_for(wl, orc, gpu, t)
        orc.step(a)
        shadow.step(a)
        gpu.step(a_dev)
        shadow.state = shadow.state.astype(np.float32).astype(np.float64)
        shadow.pid = shadow.pid.astype(np.float32).astype(np.float64)
        shadow.wind = shadow.wind.astype(np.float32).astype(np.float64)
        new_ill = shadow_drift(orc, shadow, M) & ~ill
        ill |= new_ill
        alive &= ~ill
        o64, r64, d64, margin = orc.outputs()
        o32 = gpu.obs.cpu().numpy().astype(np.float64)
        r32 = gpu.reward.cpu().numpy().astype(np.float64)
        d32 = gpu.done.cpu().numpy()
        n_done += int((d64[alive] != 0).sum())
        # done: bit-exact, threshold ties aside
        bad = alive & (d32 != d64)
        hard = bad & (margin[:, 0] >= TIE)
        assert not hard.any(), ("done mismatch", t, np.nonzero(hard)[0][:5], margin[hard][:5], d32[hard][:5], d64[hard][:5])
        ties["done"] += int(bad.sum())
        alive &= ~bad
        # reward: 1e-3 relative; the at-target indicator is a threshold too
        rerr = reward_err(r32, r64)
        bad = alive & (rerr > 1.0)
        hard = bad & (margin[:, 1] >= TIE)
        assert not hard.any(), ("reward mismatch", t, np.nonzero(hard)[0][:5], r32[hard][:5], r64[hard][:5])
        ties["reward"] += int(bad.sum())
        if over.get("reward_mode", 0) == W.REW_FLY_THROUGH:
            alive &= ~bad                                             # a capture tie also moves the target: drop the env
        worst["rew"] = max(worst["rew"], rerr[alive & ~bad].max(initial=0))
        # per-drone shares (MultiAgentAviary view): same tolerance, and they add up to the env reward
        rd64 = orc.reward_per_drone.reshape(N, M)
        rd32 = gpu.reward_per_drone.cpu().numpy().astype(np.float64).reshape(N, M)
        ok = alive & ~bad
        derr = np.abs(rd32 - rd64).max(axis=1) / (TOL_R * np.abs(rd64).max(axis=1) + R_FLOOR)   # shares: relative to the largest share of the env
        assert (derr[ok] <= 1.0).all(), ("per-drone reward mismatch", t, derr[ok].max())
        assert (np.abs(rd32.sum(axis=1) - r32)[ok] <= 1e-5 * np.maximum(1.0, np.abs(rd32).sum(axis=1))[ok]).all()
        # observation (kinematic part follows the state tolerances; adjacency is 0/1 with a threshold)
        ob32 = o32.reshape(N, M, opd)
        ob64 = o64.reshape(N, M, opd)
        if over.get("obs_mode", 0) == W.OBS_KIN20:                  # [p, q, eta, v, w, a]: q up to sign, a exact
            assert np.array_equal(ob32[alive][:, :, 16:20], ob64[alive][:, :, 16:20]), ("KIN20 action slot", t)
            dq = np.minimum(np.abs(ob32[:, :, 3:7] - ob64[:, :, 3:7]).max(axis=2), np.abs(ob32[:, :, 3:7] + ob64[:, :, 3:7]).max(axis=2))
            assert (dq[alive] <= TOL_Q).all(), ("KIN20 quaternion", t, dq[alive].max())
            ob32 = np.concatenate([ob32[:, :, 0:3], ob32[:, :, 7:16]], axis=2)
            ob64 = np.concatenate([ob64[:, :, 0:3], ob64[:, :, 7:16]], axis=2)
        if over.get("obs_mode", 0) == W.OBS_KIN12_TGT:             # the 4 target words are copied, not computed
            assert np.abs(ob32[alive][:, :, 12:16] - ob64[alive][:, :, 12:16]).max(initial=0) < 1e-6, ("KIN12_TGT target slot", t)
        if over.get("obs_mode", 0) == W.OBS_KIN12_Z:
            assert np.abs(ob32[alive][:, :, 12] - ob64[alive][:, :, 12]).max(initial=0) < 1e-6, ("KIN12_Z target altitude", t)
        if over.get("obs_mode", 0) == W.OBS_KIN12_WP:              # waypoint copied, body-frame offset follows p and q
            assert np.abs(ob32[alive][:, :, 12:15] - ob64[alive][:, :, 12:15]).max(initial=0) < 1e-6, ("KIN12_WP waypoint", t)
            assert np.abs(ob32[alive][:, :, 15:18] - ob64[alive][:, :, 15:18]).max(initial=0) < 1e-3, ("KIN12_WP body-frame offset", t)
        kin = np.abs(ob32[:, :, :12] - ob64[:, :, :12])
        kin[:, :, 3:6] = np.minimum(kin[:, :, 3:6], 2 * np.pi - kin[:, :, 3:6])     # angles wrap
        kin_tol = np.broadcast_to(np.array([TOL_P] * 3 + [2 * TOL_Q * 2] * 3 + [TOL_V] * 3 + [TOL_W] * 3), kin.shape).copy()
        # roll and yaw of the ZYX angles are ill-defined towards pitch = +-90 degrees (only their combination is fixed there):
        # d(roll), d(yaw) ~ dq / cos(pitch), so their tolerance follows 1 / cos(pitch) (a tumbling drone passes through it)
        gimbal = 1.0 / np.maximum(np.abs(np.cos(ob64[:, :, 4])), 1e-2)
        kin_tol[:, :, 3] *= gimbal
        kin_tol[:, :, 5] *= gimbal
        assert (kin[alive] <= kin_tol[alive]).all(), ("obs mismatch", t, (kin / kin_tol)[alive].max(axis=(0, 1)))
        if over.get("obs_mode", 0) == W.OBS_KIN12_ADJ:
            badadj = alive & (ob32[:, :, 12:] != ob64[:, :, 12:]).any(axis=(1, 2))
            hard = badadj & (margin[:, 2] >= TIE)
            assert not hard.any(), ("adjacency mismatch", t, np.nonzero(hard)[0][:5])
            ties["adj"] += int(badadj.sum())
        if (t + 1) % check_every == 0 or t == steps - 1:
            res, g = compare_state(orc, gpu, alive, M, f"step {t + 1}")
            for k in ("dp", "dv", "dq", "dw"):
                worst[k] = max(worst[k], res[k])
            assert np.array_equal(g["ep_step"][alive], orc.ep_step[alive]), "episode counters differ"
    n_ill = int(ill.sum())
    dropped = int((~alive & ~ill).sum())
    assert dropped <= max(2, N // 500), ("too many threshold ties", ties, dropped)
    assert n_ill <= max_ill_frac * N, ("too many ill-conditioned envs", n_ill, N)
    return dict(worst=worst, ties=ties, dropped=dropped, ill_conditioned=n_ill, n_done=n_done, kernel=gpu.kernel_name)
