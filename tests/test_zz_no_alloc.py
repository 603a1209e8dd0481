"""-m gpu: mdg_step_host_static, the host-buffer step that allocates nothing (include/mdg.h), against mdg_step_host.

Collected last on purpose (the file name): the suite runs with pytest -x, and a failure here must not hide the other tests.
The two entry points launch the same step kernel on the same actions, so the comparison is bitwise - stricter than the 1e-3 of
the parity tests.  The static staging array is shared by every handle of the process and keeps its contents between calls: the
test makes two calls in a row on one handle, then a call on a second, smaller handle (stale rows of the first stay beyond its
own), and checks the size limit's error.  It must pass alone in a fresh process and after the other tests.
"""
import numpy as np
import pytest

from paper_2606_08039_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _pair(w):
    import paper_2606_08039_b200 as mdg
    mk = lambda: mdg.Env(w.n_envs, w.n_drones, w.physics_mode, w.action_type, mdg.default_params(0, **dict(w.params, episode_len_s=3 / 48)))
    a, b = mk(), mk()
    a.reset(w.seed); b.reset(w.seed)
    return a, b


def _host_outputs(e):
    import torch
    return (torch.empty(e.n_envs * e.obs_dim, dtype=torch.float32).pin_memory(), torch.empty(e.n_envs, dtype=torch.float32).pin_memory(),
            torch.empty(e.n_envs, dtype=torch.uint8).pin_memory())


def _compare_calls(w, n_calls):
    import torch
    ref, new = _pair(w)
    if w.actions[0] == "targets":
        acts = [ref.targets.clone().cpu().pin_memory() for t in range(n_calls)]
    else:
        base = W.hover_rpm_f32() if w.actions[0] == "hover_scale" else 1.0
        acts = [ref.gen_actions(w.seed, t, base, w.actions[1], w.actions[2]).cpu().pin_memory() for t in range(n_calls)]
    torch.cuda.synchronize()
    o0, r0, d0 = _host_outputs(ref)
    o1, r1, d1 = _host_outputs(new)
    for t in range(n_calls):
        o1.fill_(float("nan")); r1.fill_(float("nan")); d1.fill_(255)
        ref.step_host(acts[t], o0, r0, d0)                       # the existing path: per-handle staging buffer (cudaMalloc on first use)
        new.step_host_static(acts[t], o1, r1, d1)                # the static array; results valid on return
        assert torch.equal(o0, o1) and torch.equal(r0, r1) and torch.equal(d0, d1), f"call {t}"
        assert torch.isfinite(o1).all() and (d1 != 255).all()
        sa, sb = ref.get_state(), new.get_state()
        for k in sa:
            assert np.array_equal(sa[k], sb[k]), (t, k)
    return new


def test_static_staging_step_equals_the_allocating_one_on_consecutive_calls():
    """Config 5 (4 drones, every aero term, VEL actions) at 5,000 envs: two calls in a row (the second finds the first call's rows
    in the array), a third that crosses an auto-reset (episodes of 3 steps), then a smaller handle of another shape whose rows
    only cover the start of the array."""
    _compare_calls(W.config(5).scaled(5000), 3)
    _compare_calls(W.config(4).scaled(37), 2)


def test_static_staging_rejects_more_drones_than_the_array_holds():
    import paper_2606_08039_b200 as mdg
    import torch
    from paper_2606_08039_b200 import binding
    w = W.config(2)
    n = binding.STATIC_STAGE_MAX_DRONES + 1
    big = mdg.Env(n, 1, w.physics_mode, w.action_type, mdg.default_params(0, **w.params))
    big.reset(w.seed)
    acts = torch.zeros(n * 4, dtype=torch.float32)
    with pytest.raises(mdg.MdgError) as exc:
        big.step_host_static(acts)
    assert str(binding.STATIC_STAGE_MAX_DRONES) in str(exc.value) and str(n) in str(exc.value)
    ok = mdg.Env(binding.STATIC_STAGE_MAX_DRONES, 1, w.physics_mode, w.action_type, mdg.default_params(0, **w.params))
    ok.reset(w.seed)
    ok.step_host_static(torch.zeros(binding.STATIC_STAGE_MAX_DRONES * 4, dtype=torch.float32))   # exactly the limit is accepted
