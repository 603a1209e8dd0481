"""-m gpu: seeded random SEQUENCES of API calls on one handle against a second handle that only ever makes plain, synchronised
mdg_step calls - bitwise.

Every way of advancing the simulation (mdg_step, mdg_step_chained, mdg_step_many as a replayed graph, mdg_step_host,
mdg_step_host_static) computes the same step; what differs is the scheduling around it (item-level chaining, the smaller grid of
chained launches, ticket dispensers taking turns, graph replays with baked launch numbers, stream changes, checkpoints).  The
sequences interleave them with resets, a checkpoint restored into a fresh handle, stream switches and camera calls, on a batch
that fills the device (two envs per lane, dispensers in use) and on one that does not (one work item per warp).
"""
import random

import numpy as np
import pytest

from paper_2606_08039_b200 import workloads as W

pytestmark = pytest.mark.gpu


def same(a, b, what):
    import torch
    sa, sb = a.get_state(), b.get_state()
    for k in sa:
        assert np.array_equal(sa[k], sb[k]), (what, k)
    assert torch.equal(a.obs, b.obs) and torch.equal(a.reward, b.reward) and torch.equal(a.done, b.done), what
    assert torch.equal(a.reward_per_drone, b.reward_per_drone) and torch.equal(a.targets, b.targets), what


@pytest.mark.parametrize("c,n_envs,seed", [(5, 40003, 1), (5, 40003, 2), (3, 3001, 3), (4, 257, 4), (5, 40003, 5), (2, 70001, 6)])
def test_random_call_sequences_equal_plain_stepping(c, n_envs, seed):
    import torch
    import paper_2606_08039_b200 as mdg
    rng = random.Random(seed)
    wl = W.config(c).scaled(n_envs)
    over = dict(wl.params, episode_len_s=9 / 48)                  # auto-resets every nine steps
    mk = lambda: mdg.Env(wl.n_envs, wl.n_drones, wl.physics_mode, wl.action_type, mdg.default_params(0, **over))
    fancy, plain = mk(), mk()
    fancy.reset(wl.seed); plain.reset(wl.seed)
    base = W.hover_rpm_f32() if wl.actions[0] == "hover_scale" else 1.0
    A = 16
    if wl.actions[0] == "targets":                                # PID waypoints: any fixed rows serve, both handles get the same
        acts = [plain.targets.clone() + 0.01 * t for t in range(A)]
    else:
        acts = [plain.gen_actions(wl.seed, t, base, wl.actions[1], wl.actions[2]) for t in range(A)]
    stack = torch.stack(acts)                                     # [A, D, 4] for mdg_step_many
    host = [a.cpu().pin_memory() for a in acts]
    torch.cuda.synchronize()
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    t = 0
    log = []
    for op_i in range(70):
        op = rng.choice(["step", "chained", "chained", "chained", "many", "host", "static", "reset", "ckpt", "stream", "render", "chained_burst"])
        log.append(op)
        if op in ("step", "chained"):
            (fancy.step if op == "step" else fancy.step_chained)(acts[t % A]); plain.step(acts[t % A]); t += 1
        elif op == "chained_burst":
            n = rng.choice([2, 5, 13])
            for _ in range(n):
                fancy.step_chained(acts[t % A]); plain.step(acts[t % A]); t += 1
        elif op == "many":
            n = rng.choice([2, 3, 4])
            k0 = t % A
            if k0 + n > A:
                continue
            for rep in range(rng.choice([1, 2])):                 # replays of the cached graph
                fancy.step_many(stack[k0:k0 + n], n)
                for k in range(n):
                    plain.step(acts[k0 + k])
            t = k0 + n
        elif op in ("host", "static"):
            torch.cuda.synchronize()
            (fancy.step_host if op == "host" else fancy.step_host_static)(host[t % A]); plain.step(acts[t % A]); t += 1
        elif op == "reset":
            s = rng.randrange(1 << 30)
            fancy.reset(s); plain.reset(s)
        elif op == "ckpt":
            torch.cuda.synchronize()
            blob = fancy.save()
            fresh = mk()
            fresh.load(blob)
            fancy = fresh
        elif op == "stream":
            torch.cuda.synchronize()                              # the actions were produced on the default stream
            fancy.set_stream(rng.choice(streams))
        elif op == "render":
            fancy.render_depth(); fancy.render_rgba()
        if op_i % 10 == 9:
            torch.cuda.synchronize()
            same(fancy, plain, (seed, op_i, log[-12:]))
    torch.cuda.synchronize()
    same(fancy, plain, (seed, "end", log[-12:]))
