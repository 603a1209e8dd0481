"""The N>1 path on CPU (gloo, world_size 2): env-range sharding with env_index_base reproduces the
unsplit batch exactly (no collective on the step path), and the timing reduction is a max over ranks."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2606_08039_b200 import workloads as W
from paper_2606_08039_b200.sharding import max_over_ranks, replica_base, shard_range


def test_shard_ranges_tile_the_batch():
    for n, w in ((65536, 8), (10, 3), (7, 7), (1001, 4)):
        spans = [shard_range(n, r, w) for r in range(w)]
        assert spans[0][0] == 0 and sum(c for _, c in spans) == n
        for (b0, c0), (b1, _) in zip(spans, spans[1:]):
            assert b0 + c0 == b1
    assert replica_base(2, 1, 4, 100) == 900


def _worker(rank, world, port, n_total, steps, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from oracle import oracle as O
    wl = W.config(5)
    base, cnt = shard_range(n_total, rank, world)
    env = O.OracleEnv(cnt, wl.n_drones, wl.physics_mode, wl.action_type,
                      O.OracleParams(0, **dict(wl.params, env_index_base=base, episode_len_s=5 / 48)))
    env.reset(wl.seed)
    for t in range(steps):
        env.step(O.gen_actions(wl.seed, t, cnt, wl.n_drones, 1.0, -1.0, 1.0, env_base=base))
    obs, rew, done, _ = env.outputs()
    parts = [None] * world
    dist.all_gather_object(parts, (base, env.state, obs, rew, done))       # test plumbing only
    slowest = max_over_ranks(10.0 + rank, dist)
    if rank == 0:
        parts.sort(key=lambda p: p[0])
        np.savez(out, state=np.concatenate([p[1] for p in parts]), obs=np.concatenate([p[2] for p in parts]),
                 rew=np.concatenate([p[3] for p in parts]), done=np.concatenate([p[4] for p in parts]), slowest=slowest)
    dist.destroy_process_group()


def test_two_rank_sharding_matches_the_unsplit_batch(tmp_path):
    from oracle import oracle as O
    n_total, steps, world = 37, 10, 2
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    out = str(tmp_path / "gathered.npz")
    mp.spawn(_worker, args=(world, port, n_total, steps, out), nprocs=world, join=True)
    got = np.load(out)
    wl = W.config(5)
    env = O.OracleEnv(n_total, wl.n_drones, wl.physics_mode, wl.action_type, O.OracleParams(0, **dict(wl.params, episode_len_s=5 / 48)))
    env.reset(wl.seed)
    for t in range(steps):
        env.step(O.gen_actions(wl.seed, t, n_total, wl.n_drones, 1.0, -1.0, 1.0))
    obs, rew, done, _ = env.outputs()
    assert np.array_equal(got["state"], env.state) and np.array_equal(got["obs"], obs)
    assert np.array_equal(got["rew"], rew) and np.array_equal(got["done"], done) and done.any()
    assert float(got["slowest"]) == 11.0
