"""-m gpu: the CUDA path (through the C ABI) against the float64 oracle on the five BASELINE.json
configs, 48 control steps = 1 s of simulated time, plus feature-by-feature and edge cases."""
import os

import numpy as np
import pytest

from paper_2606_08039_b200 import workloads as W
from parity_util import run_parity

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("c", [1, 2, 3, 4])
def test_config_parity_full_size(c):
    # c4: close downwash passes are chaotic (parity_util "Conditioning"); measured 13 of 1,024 envs on the fixed seed, cap = 2 x that
    res = run_parity(W.config(c), steps=48, max_ill_frac=26 / 1024 if c == 4 else 0.0)
    print(c, res)
    assert "generic" not in res["kernel"]


def test_config5_parity_sampled_size():
    """c5 at 4,099 envs (several blocks and a ragged tail); the full 65,536 x 4 run is the next test."""
    res = run_parity(W.config(5).scaled(4099), steps=48)
    print(res)
    assert "generic" not in res["kernel"]


def test_config5_parity_full_size():
    res = run_parity(W.config(5), steps=48, check_every=16)
    print(res)


@pytest.mark.parametrize("c", [1, 2, 3, 4, 5])
def test_config_parity_with_frequent_episodes(c):
    """Short episodes + crashes: exercises truncation, termination and same-call auto-reset every few steps."""
    wl = W.config(c).scaled(min(W.config(c).n_envs, 1500))
    res = run_parity(wl, steps=40, extra=dict(episode_len_s=7 / 48, z_max=1.3), max_ill_frac=0.0)   # measured: no ill-conditioned env in any config
    print(c, res)
    assert res["n_done"] > wl.n_envs


@pytest.mark.parametrize("c,extra", [(3, dict(term_dist=1.06)), (4, dict(z_max=1.0)), (5, dict(term_dist=0.35))])
def test_config_parity_with_divergent_resets(c, extra):
    """Envs that terminate one by one at different steps: neighbouring envs of one warp take the auto-reset path at
    different times (the truncation test above resets whole warps at once)."""
    wl = W.config(c).scaled(min(W.config(c).n_envs, 2051))
    res = run_parity(wl, steps=48, extra=extra, max_ill_frac=10 / 1024 if c == 4 else 0.0)      # c4: measured 5 of 1,024, cap = 2 x that
    print(c, res)
    assert res["n_done"] > wl.n_envs // 8


# Measured with the oracle alone on the fixed seeds (the exclusion depends on nothing else): c4 13 ill-conditioned + 200 envs that
# came within 1e-4 of a threshold (mostly floor contacts), 210 distinct; c3 and c5: none.  Cap = 2 x ill + near-threshold.
MAX_EXCLUDED = {5: 0, 4: 226, 3: 0}


@pytest.mark.parametrize("c,n_envs", [(5, 65536), (4, 1024), (3, 16384)])
def test_back_to_back_steps_without_host_sync(c, n_envs):
    """48 steps queued back to back (no host read in between): consecutive launches overlap through programmatic
    dependent launch and per-item sequence flags, so this is the test of that dependency chain.  The end state,
    the last outputs and the episode counters must match the oracle as in the step-by-step tests."""
    import torch
    from oracle import oracle as O
    from parity_util import make_pair, compare_state, shadow_drift, reward_err
    wl = W.config(c).scaled(n_envs)
    orc, gpu = make_pair(wl)
    shadow = O.OracleEnv(wl.n_envs, wl.n_drones, wl.physics_mode, wl.action_type, O.OracleParams(0, **wl.params), n_threads=os.cpu_count() or 1)
    for s in (orc, shadow, gpu):
        s.reset(wl.seed)
    steps = 48
    if wl.actions[0] == "targets":
        acts = [orc.targets.astype(np.float32)] * steps
        dev = [torch.from_numpy(acts[0]).cuda()] * steps
    else:
        base = W.hover_rpm_f32() if wl.actions[0] == "hover_scale" else 1.0
        acts = [O.gen_actions(wl.seed, t, wl.n_envs, wl.n_drones, base, wl.actions[1], wl.actions[2]) for t in range(steps)]
        dev = [gpu.gen_actions(wl.seed, t, base, wl.actions[1], wl.actions[2]) for t in range(steps)]
    torch.cuda.synchronize()
    for t in range(steps):                       # nothing but launches; the actions were all there before the first one
        gpu.step_chained(dev[t])
    ill = np.zeros(wl.n_envs, dtype=bool)
    differ = np.zeros(wl.n_envs, dtype=bool)     # envs whose done history may legitimately differ (threshold ties)
    for t in range(steps):
        orc.step(acts[t])
        shadow.step(acts[t])
        shadow.state = shadow.state.astype(np.float32).astype(np.float64)
        shadow.pid = shadow.pid.astype(np.float32).astype(np.float64)
        shadow.wind = shadow.wind.astype(np.float32).astype(np.float64)
        ill |= shadow_drift(orc, shadow, wl.n_drones)
        differ |= orc.outputs()[3][:, 0] < 1e-4
    torch.cuda.synchronize()
    alive = ~ill & ~differ
    # envs left out: ill-conditioned downwash passes (shadow oracle, c4 only) + envs that came within 1e-4 of a termination threshold
    # at any of the 48 steps (their done history may legitimately differ).
    print(c, "excluded", int((~alive).sum()), "of", wl.n_envs, "ill", int(ill.sum()), "near-threshold", int(differ.sum()))
    assert (~alive).sum() <= MAX_EXCLUDED[c], (int(ill.sum()), int(differ.sum()))
    res, g = compare_state(orc, gpu, alive, wl.n_drones, "after 48 queued steps")
    print(c, res, int((~alive).sum()))
    assert np.array_equal(g["ep_step"][alive], orc.ep_step[alive])
    _, r64, d64, _ = orc.outputs()
    assert np.array_equal(gpu.done.cpu().numpy()[alive], d64[alive])
    rerr = reward_err(gpu.reward.cpu().numpy().astype(np.float64), r64)
    margin = orc.outputs()[3]
    assert (rerr[alive & (margin[:, 1] >= 1e-4)] <= 1.0).all(), rerr[alive].max()      # every reward, at-target threshold ties aside


def test_interleaved_handles_and_host_step_are_bitwise_the_plain_sequence():
    """bench.py's pattern: several handles stepped round-robin on one stream with nothing in between (each launch chains
    on its own handle's previous step, the kernels of different handles overlap).  Results must equal, bit for bit, the
    same handles stepped one at a time with a host sync after every step; mdg_step_host must equal mdg_step."""
    import torch
    import paper_2606_08039_b200 as mdg
    wl = W.config(5).scaled(20000)                              # saturating grid: the chained path is taken
    def make(k):
        e = mdg.Env(wl.n_envs, wl.n_drones, wl.physics_mode, wl.action_type, mdg.default_params(0, **dict(wl.params, env_index_base=k * wl.n_envs)))
        e.reset(wl.seed + k)
        return e
    fast, slow = [make(k) for k in range(3)], [make(k) for k in range(3)]
    host = make(0)
    acts = [[fast[k].gen_actions(wl.seed + k, t, 1.0, -1.0, 1.0) for t in range(24)] for k in range(3)]
    torch.cuda.synchronize()
    for t in range(24):
        for k in range(3):
            fast[k].step_chained(acts[k][t])
    for t in range(24):
        for k in range(3):
            slow[k].step(acts[k][t])
            torch.cuda.synchronize()
    obs_h = torch.empty((wl.n_envs, host.obs_dim), dtype=torch.float32).pin_memory()
    rew_h = torch.empty(wl.n_envs, dtype=torch.float32).pin_memory()
    done_h = torch.empty(wl.n_envs, dtype=torch.uint8).pin_memory()
    for t in range(24):
        host.step_host(acts[0][t].cpu().pin_memory(), obs_h, rew_h, done_h)
    torch.cuda.synchronize()
    for k in range(3):
        a, b = fast[k].get_state(), slow[k].get_state()
        for key in ("state", "ctrl", "targets", "wind", "ep_step"):
            assert np.array_equal(a[key], b[key]), (k, key)
        assert torch.equal(fast[k].obs, slow[k].obs) and torch.equal(fast[k].reward, slow[k].reward) and torch.equal(fast[k].done, slow[k].done)
    assert np.array_equal(host.get_state()["state"], slow[0].get_state()["state"])
    assert torch.equal(obs_h, slow[0].obs.cpu().reshape(wl.n_envs, -1)) and torch.equal(rew_h, slow[0].reward.cpu()) and torch.equal(done_h, slow[0].done.cpu())
