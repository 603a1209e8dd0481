"""-m gpu: stream, graph and sharding semantics of the CUDA path (through the C ABI).

* mdg_step has plain stream semantics: an in-stream producer (mdg_gen_actions, a torch kernel) may write the action buffer
  right before it, with no host synchronisation anywhere (the RL loop of PAPER.md:285-292).
* mdg_step_chained / mdg_step_many overlap consecutive steps; their results are bitwise those of synchronised single steps,
  also when a replay follows mdg_load.
* A batch split into shards with env_index_base draws what the whole batch draws (the PRNG key is part of the
  state): two CUDA handles concatenated are bitwise one handle, and each matches the oracle's shard.
* Distinct handles are independent: two host threads drive two handles through mdg_step_host at the same time.
"""
import os
import threading

import numpy as np
import pytest

from paper_2606_08039_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _mk(w, **over):
    import paper_2606_08039_b200 as mdg
    return mdg.Env(w.n_envs, w.n_drones, w.physics_mode, w.action_type, mdg.default_params(0, **dict(w.params, **over)))


def _same(a, b, what=""):
    import torch
    sa, sb = a.get_state(), b.get_state()
    for k in sa:
        assert np.array_equal(sa[k], sb[k]), (what, k)
    assert torch.equal(a.obs, b.obs) and torch.equal(a.reward, b.reward) and torch.equal(a.done, b.done), what
    assert torch.equal(a.reward_per_drone, b.reward_per_drone), what


@pytest.mark.parametrize("producer", ["mdg_gen_actions", "torch_kernel"])
def test_in_stream_producer_between_steps_needs_no_host_sync(producer):
    """48 c5 steps at 20,000 envs (a grid that fills the device); each step's actions are written into ONE reused buffer by a
    kernel enqueued between the steps, nothing synchronises the host.  Must equal, bit for bit, the synchronised sequence."""
    import torch
    w = W.config(5).scaled(20000)
    fast, slow = _mk(w, episode_len_s=11 / 48), _mk(w, episode_len_s=11 / 48)
    fast.reset(w.seed); slow.reset(w.seed)
    pre = [slow.gen_actions(w.seed, t, 1.0, -1.0, 1.0) for t in range(48)]
    torch.cuda.synchronize()
    buf = torch.empty_like(pre[0])
    for t in range(48):
        if producer == "mdg_gen_actions":
            fast.gen_actions(w.seed, t, 1.0, -1.0, 1.0, out=buf)
        else:
            torch.mul(pre[t], 1.0, out=buf)              # an elementwise torch kernel on the same stream
        fast.step(buf)
    for t in range(48):
        slow.step(pre[t])
        torch.cuda.synchronize()
    _same(fast, slow, producer)


def test_graph_replay_chains_and_equals_single_steps_also_after_load():
    """mdg_step_many: 48 c5 steps as one CUDA graph (inner launches chained item by item), replayed twice, then again after
    mdg_load of an earlier checkpoint and after a reset with another seed (graph rebuilt); always bitwise the single steps."""
    import torch
    w = W.config(5).scaled(20000)
    a, b = _mk(w, episode_len_s=17 / 48), _mk(w, episode_len_s=17 / 48)
    a.reset(w.seed); b.reset(w.seed)
    acts = torch.stack([a.gen_actions(w.seed, t, 1.0, -1.0, 1.0) for t in range(48)])
    torch.cuda.synchronize()
    for rep in range(2):
        for t in range(48):
            a.step(acts[t])
            torch.cuda.synchronize()
        b.step_many(acts, 48)
        _same(a, b, f"replay {rep}")
    blob = a.save()
    for t in range(5):
        a.step(acts[t]); b.step_chained(acts[t])
    _same(a, b, "chained steps after a replay")
    a.load(blob); b.load(blob)
    for t in range(48):
        a.step(acts[t])
    b.step_many(acts, 48)
    _same(a, b, "replay after mdg_load")
    a.reset(99); b.reset(99)
    for t in range(48):
        a.step(acts[t])
    b.step_many(acts, 48)
    _same(a, b, "replay after reset with another seed")
    # a small grid (one warp per item, no ticket dispenser) through the same path
    w3 = W.config(3).scaled(3000)
    c, d = _mk(w3), _mk(w3)
    c.reset(w3.seed); d.reset(w3.seed)
    tg = torch.stack([c.targets.clone()] * 12)
    for t in range(12):
        c.step(tg[t])
    d.step_many(tg, 12)
    _same(c, d, "small-grid replay")


def test_cuda_shards_concatenate_bitwise_to_the_whole_batch_and_match_the_oracle_shards():
    """(env_index_base 0, n 1,500) || (1,500, n 2,599) == one handle of 4,099 envs, bit for bit, after 48 c5 steps with
    auto-resets every 7 steps: state, controller memory, targets, wind, counters, obs, reward, done."""
    import torch
    from oracle import oracle as O
    from parity_util import TOL_P, TOL_V, TOL_Q, reward_err
    w = W.config(5).scaled(4099)
    over = dict(episode_len_s=7 / 48)
    whole = _mk(w, **over)
    parts = [(0, 1500), (1500, 2599)]
    shards = [_mk(w.scaled(n), env_index_base=b, **over) for b, n in parts]
    orcs = [O.OracleEnv(n, w.n_drones, w.physics_mode, w.action_type, O.OracleParams(0, **dict(w.params, env_index_base=b, **over)),
                        n_threads=os.cpu_count() or 1) for b, n in parts]
    for e in [whole] + shards + orcs:
        e.reset(w.seed)
    M = w.n_drones
    for t in range(48):
        a = whole.gen_actions(w.seed, t, 1.0, -1.0, 1.0)
        whole.step(a)
        for (b, n), sh, orc in zip(parts, shards, orcs):
            a_sh = sh.gen_actions(w.seed, t, 1.0, -1.0, 1.0)
            assert torch.equal(a_sh, a[b * M:(b + n) * M])              # the harness stream is keyed on the global env index too
            sh.step(a_sh)
            orc.step(a_sh.cpu().numpy())
    torch.cuda.synchronize()
    sw = whole.get_state()
    ss = [s.get_state() for s in shards]
    for k in sw:
        assert np.array_equal(sw[k], np.concatenate([s[k] for s in ss])), k
    for name in ("obs", "reward", "done", "reward_per_drone"):
        assert torch.equal(getattr(whole, name), torch.cat([getattr(s, name) for s in shards])), name
    for sh, orc, st in zip(shards, orcs, ss):                           # and each CUDA shard against the oracle's shard
        s64, s32 = orc.state, st["state"].astype(np.float64)
        _, r64, d64, margin = orc.outputs()
        ok = np.repeat(margin[:, 0] >= 1e-4, M)
        assert np.abs(s32[:, 0:3] - s64[:, 0:3])[ok].max() <= TOL_P and np.abs(s32[:, 7:10] - s64[:, 7:10])[ok].max() <= TOL_V
        dq = np.minimum(np.abs(s32[:, 3:7] - s64[:, 3:7]).max(axis=1), np.abs(s32[:, 3:7] + s64[:, 3:7]).max(axis=1))
        assert dq[ok].max() <= TOL_Q
        assert np.array_equal(st["ep_step"], orc.ep_step)
        okr = (margin[:, 0] >= 1e-4) & (margin[:, 1] >= 1e-4)
        assert np.array_equal(sh.done.cpu().numpy()[okr], d64[okr])
        assert (reward_err(sh.reward.cpu().numpy().astype(np.float64), r64)[okr] <= 1.0).all()


def test_two_host_threads_drive_two_handles_through_the_host_call():
    """include/mdg.h: distinct handles are independent.  Two threads, each with its own handle and stream, 1,000 mdg_step_host
    calls each; the results equal those of two fresh handles driven one after the other."""
    import torch
    w = W.config(5).scaled(512)
    n_it = 1000

    def make():
        envs = [_mk(w, env_index_base=k * w.n_envs) for k in range(2)]
        for k, e in enumerate(envs):
            e.set_stream(torch.cuda.Stream())
            e.reset(w.seed + k)
        return envs

    threaded, sequential = make(), make()
    acts = [[threaded[k].gen_actions(w.seed + k, t, 1.0, -1.0, 1.0).cpu().pin_memory() for t in range(8)] for k in range(2)]
    torch.cuda.synchronize()
    errors = []

    def drive(env, a):
        try:
            obs = torch.empty((w.n_envs, env.obs_dim)).pin_memory()
            rew, done = torch.empty(w.n_envs).pin_memory(), torch.empty(w.n_envs, dtype=torch.uint8).pin_memory()
            for t in range(n_it):
                env.step_host(a[t % 8], obs, rew, done)
        except Exception as exc:                                              # pragma: no cover
            errors.append(exc)

    th = [threading.Thread(target=drive, args=(threaded[k], acts[k])) for k in range(2)]
    for t in th:
        t.start()
    for t in th:
        t.join()
    for k in range(2):
        drive(sequential[k], acts[k])
    assert not errors, errors
    torch.cuda.synchronize()
    for k in range(2):
        _same(threaded[k], sequential[k], f"thread {k}")


def test_failed_run_time_specialisation_is_reported_and_require_mode_fails(monkeypatch):
    """No csrc/ sources (MDG_JIT_SRC points nowhere): a feature word without a precompiled instance falls back to the generic
    kernel, says so in mdg_last_error(), and fails outright under MDG_JIT=require."""
    import paper_2606_08039_b200 as mdg
    over = dict(obs_noise=[0.0, 0.031, 0.0, 0.0])                             # a feature word of its own (cache key: the word, not the values)
    w = W.config(2).scaled(256)
    monkeypatch.setenv("MDG_JIT_SRC", "/nonexistent/csrc")
    # another G than any other test uses with this word, so the per-process cache cannot hold a compiled instance
    e = mdg.Env(w.n_envs, 3, w.physics_mode, w.action_type, mdg.default_params(0, **dict(w.params, **over)))
    assert "generic" in e.kernel_name
    note = mdg.lib().mdg_last_error().decode()
    assert "generic kernel" in note and "NVRTC" in note, note
    monkeypatch.setenv("MDG_JIT", "require")
    with pytest.raises(mdg.MdgError) as exc:
        mdg.Env(w.n_envs, 3, w.physics_mode, w.action_type, mdg.default_params(0, **dict(w.params, **over)))
    assert "require" in str(exc.value)
    monkeypatch.delenv("MDG_JIT_SRC")
    monkeypatch.setenv("MDG_JIT", "1")
    ok = mdg.Env(w.n_envs, 5, w.physics_mode, w.action_type, mdg.default_params(0, **dict(w.params, **over)))
    assert "jit" in ok.kernel_name and mdg.lib().mdg_last_error().decode() == ""
