"""Host-side sharding helpers: envs are independent, so a batch is split into
contiguous env ranges, one per GPU / process, with NO collective on the step path.  Philox counters use
`env_index_base + e`, so every shard draws exactly what the unsplit batch would.  The only cross-rank
operation is the max-over-ranks of the timed region (bench.py)."""


def shard_range(n_envs_total: int, rank: int, world: int):
    """Contiguous range of rank: (env_index_base, n_envs); ranges tile [0, n_envs_total) without gaps."""
    if not (0 <= rank < world) or n_envs_total < world:
        raise ValueError("need 0 <= rank < world <= n_envs_total")
    q, r = divmod(n_envs_total, world)
    base = rank * q + min(rank, r)
    return base, q + (1 if rank < r else 0)


def replica_base(rank: int, replica: int, n_replicas: int, n_envs: int) -> int:
    """Weak scaling (bench.py): rank r, replica k simulates envs [base, base + n_envs)."""
    return (rank * n_replicas + replica) * n_envs


def max_over_ranks(value: float, dist=None, device=None) -> float:
    """Max of a per-rank scalar (elapsed ms) over the process group; identity without a group."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
