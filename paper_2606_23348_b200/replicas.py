"""Host-side logic of the multi-GPU mode: replicas over disjoint global game-id ranges.

Games are independent (PAPER.md P:L118 batched envs, P:L61 no cross-game coupling), so the path has
no exchange step and no collective.  Every random draw is keyed by the global
game id = game_id_base + g, hence any partition reproduces the single-GPU result bit for bit.
This module holds only the partition arithmetic and the timing reduction bench.py uses.
"""


def weak_replica_config(cfg, rank):
    """Weak scaling (bench.py --gpus N): every rank runs cfg['n_games'] games of its own, ids
    [rank*n, (rank+1)*n) above the configured base."""
    out = dict(cfg)
    out["game_id_base"] = int(cfg.get("game_id_base", 0)) + rank * int(cfg["n_games"])
    if out["game_id_base"] + out["n_games"] > 1 << 32:
        raise ValueError("global game ids must fit 32 bits")
    return out


def strong_replica_config(cfg, rank, world):
    """Strong scaling: cfg['n_games'] games in total, split into contiguous ranges whose sizes
    differ by at most one (the first n % world ranks take one more)."""
    n = int(cfg["n_games"])
    q, r = divmod(n, world)
    lo = rank * q + min(rank, r)
    out = dict(cfg)
    out["n_games"] = q + (1 if rank < r else 0)
    out["game_id_base"] = int(cfg.get("game_id_base", 0)) + lo
    return out


def max_over_ranks(value, dist=None, device=None):
    """Device time of the job = the slowest rank's (bench contract).  `dist` is torch.distributed
    when a process group is up, else None (single process)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
