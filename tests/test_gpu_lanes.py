"""-m gpu: the two-envs-per-lane instantiation of the step kernel (packed FP32 pairs in the substep loop).

Both instantiations are written over one lane-generic substep, every operation spelled out, so they must agree BIT FOR BIT:
the packed kernel is checked against the one-env-per-lane kernel on the same inputs (which the other test files check against
the oracle), and directly against the oracle where it is the default (config 5 at full size, tests/test_gpu_parity.py).
MDG_LANES=1|2 forces the choice (default: 2 when the grid still fills the device with half the warps).
"""
import numpy as np
import pytest

from paper_2606_08039_b200 import workloads as W
import test_gpu_features as F

pytestmark = pytest.mark.gpu


def _mk(monkeypatch, w, lanes, model=0, **over):
    import paper_2606_08039_b200 as mdg
    monkeypatch.setenv("MDG_LANES", str(lanes))
    e = mdg.Env(w.n_envs, w.n_drones, w.physics_mode, w.action_type, mdg.default_params(model, **dict(w.params, **over)))
    monkeypatch.delenv("MDG_LANES")
    return e


def _actions(w, env, t):
    if w.actions[0] == "targets":
        return env.targets.clone()
    return env.gen_actions(w.seed, t, W.hover_rpm_f32() if w.actions[0] == "hover_scale" else 1.0, w.actions[1], w.actions[2])


def _assert_same(a, b, what):
    import torch
    sa, sb = a.get_state(), b.get_state()
    for k in sa:
        assert np.array_equal(sa[k], sb[k]), (what, k)
    for name in ("obs", "reward", "done", "reward_per_drone"):
        assert torch.equal(getattr(a, name), getattr(b, name)), (what, name)


def _run_pair(monkeypatch, w, steps=48, prepare=None, **over):
    import torch
    one, two = _mk(monkeypatch, w, 1, **over), _mk(monkeypatch, w, 2, **over)
    assert ",x2>" in two.kernel_name and ",x2>" not in one.kernel_name, (one.kernel_name, two.kernel_name)
    one.reset(w.seed); two.reset(w.seed)
    if prepare:
        prepare(one); prepare(two)
    for t in range(steps):
        a = _actions(w, one, t)
        one.step(a); two.step(a)
        if t % 12 == 11:
            torch.cuda.synchronize()
            _assert_same(one, two, (w.name, t))
    torch.cuda.synchronize()
    _assert_same(one, two, (w.name, "end"))
    return one, two


@pytest.mark.parametrize("c,n", [(1, 1), (1, 77), (2, 4096), (3, 16384), (4, 1024), (5, 4099), (5, 65536)])
def test_two_lanes_equal_one_lane_on_the_configs(c, n, monkeypatch):
    """The five BASELINE.json configs (full size, and ragged sizes: an odd env count leaves the second env slot of the last item empty)."""
    _run_pair(monkeypatch, W.config(c).scaled(n), steps=48 if n < 60000 else 24)


@pytest.mark.parametrize("c", [3, 4, 5])
def test_two_lanes_equal_one_lane_with_frequent_and_divergent_resets(c, monkeypatch):
    """Auto-resets in one env slot of a lane but not in the other, every few steps."""
    w = W.config(c).scaled(min(W.config(c).n_envs, 2051))
    _run_pair(monkeypatch, w, steps=40, episode_len_s=7 / 48, z_max=1.3)
    _run_pair(monkeypatch, w, steps=48, **{3: dict(term_dist=1.06), 4: dict(z_max=1.0), 5: dict(term_dist=0.35)}[c])


CAPABLE = [k for k in sorted(F.CASES) if not any(x in k for x in ("latency", "motor_lag"))]


@pytest.mark.parametrize("name", CAPABLE)
def test_two_lanes_equal_one_lane_on_every_feature_case(name, monkeypatch):
    """Every generic-kernel case whose rotor commands stay fixed over a step (no motor lag, no latency rows), through the
    run-time instantiation of its feature word in both shapes: partial lane groups, DYN, DR planes, sensors, wind mixes,
    waypoint tasks, the moving formation centre."""
    w, extra = F.CASES[name]
    _run_pair(monkeypatch, w, steps=36, **extra)


def test_lag_and_latency_rows_stay_on_one_lane(monkeypatch):
    w, extra = F.CASES["m4_latency_motor_lag_dr"]
    e = _mk(monkeypatch, w, 2, **extra)
    assert ",x2>" not in e.kernel_name


def test_fast_spins_take_the_exact_path_in_both_shapes(monkeypatch):
    """Body rates beyond the series' range (|omega| h > 0.28 rad for controller actions, 0.75 rad otherwise): the packed kernel
    redoes the item with the one-env code, so the two shapes still agree bit for bit, and both follow the oracle."""
    import torch
    from oracle import oracle as O
    from parity_util import TOL_P, TOL_Q, TOL_V, TOL_W
    for c, spin in ((5, 90.0), (2, 260.0)):
        w = W.config(c).scaled(1500)
        over = dict(term_mode=W.TERM_NONE, auto_reset=0, episode_len_s=0.0)

        def prepare(env, spin=spin):
            st = env.get_state()["state"]
            rng = np.random.default_rng(5)
            fast = rng.uniform(size=st.shape[0]) < 0.3                  # a third of the drones, scattered over both env slots
            st[fast, 10:13] = rng.uniform(-1, 1, (int(fast.sum()), 3)).astype(np.float32) * spin
            env.set_state(state=st)

        one, two = _run_pair(monkeypatch, w, steps=6, prepare=prepare, **over)
        orc = O.OracleEnv(w.n_envs, w.n_drones, w.physics_mode, w.action_type, O.OracleParams(0, **dict(w.params, **over)), n_threads=8)
        orc.reset(w.seed)
        probe = _mk(monkeypatch, w, 1, **over)
        probe.reset(w.seed); prepare(probe)
        orc.state = probe.get_state()["state"].astype(np.float64)
        for t in range(2):                                                  # the spin decays quickly under drag / control: compare early
            a = _actions(w, probe, t)
            probe.step(a); orc.step(a.cpu().numpy())
        torch.cuda.synchronize()
        s32, s64 = probe.get_state()["state"].astype(np.float64), orc.state
        assert np.abs(s64[:, 10:13]).max() > 0.28 * 240 / 2                  # still spinning fast in the oracle
        assert np.abs(s32[:, 0:3] - s64[:, 0:3]).max() <= TOL_P and np.abs(s32[:, 7:10] - s64[:, 7:10]).max() <= TOL_V
        dq = np.minimum(np.abs(s32[:, 3:7] - s64[:, 3:7]).max(axis=1), np.abs(s32[:, 3:7] + s64[:, 3:7]).max(axis=1))
        assert dq.max() <= TOL_Q and np.abs(s32[:, 10:13] - s64[:, 10:13]).max() <= 20 * TOL_W   # rates of 100-260 rad/s: relative 1e-4
