"""Multi-GPU mode = replicas over disjoint global game-id ranges: the host-side
partition logic under a world-size-2 gloo group on CPU.  The oracle stands in for the engine (this is
a CPU test); what is checked is that the partition reproduces the one-process result bit for bit
(metamorphic pin M2) and that the timing reduction takes the max over ranks."""
import os
import socket

import numpy as np
import pytest
import torch.distributed as dist
import torch.multiprocessing as mp

import workloads
from paper_2606_23348_b200 import replicas

FIELDS = ["army", "owner", "terrain", "turn", "episode", "alive", "land", "army_total", "obs_digest",
          "episodes_done", "wins"]
STEPS = 40


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _run_oracle(cfg):
    from oracle import oracle
    o = oracle.Oracle(cfg)
    o.reset()
    for _ in range(STEPS):
        o.step()
    return {f: np.array(o.field(f), copy=True) for f in FIELDS}


def _worker(rank, world, port, mode, cfg, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        mine = (replicas.weak_replica_config(cfg, rank) if mode == "weak"
                else replicas.strong_replica_config(cfg, rank, world))
        res = _run_oracle(mine)
        slowest = replicas.max_over_ranks(10.0 + rank, dist)
        dist.barrier()
        np.savez(os.path.join(out_dir, f"r{rank}.npz"), slowest=slowest, base=mine["game_id_base"],
                 n=mine["n_games"], **res)
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("mode,n", [("weak", 24), ("strong", 37)])
def test_two_replicas_equal_one_process(tmp_path, oracle_mod, mode, n):
    cfg, _ = workloads.config("c2_24x24", n_games=n, max_turns=30, game_id_base=1000)
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), mode, cfg, str(tmp_path)), nprocs=world, join=True)
    parts = [np.load(tmp_path / f"r{r}.npz") for r in range(world)]
    total = n * world if mode == "weak" else n
    whole = _run_oracle(dict(cfg, n_games=total))
    assert [int(p["base"]) for p in parts] == [1000, 1000 + int(parts[0]["n"])]
    assert sum(int(p["n"]) for p in parts) == total
    for f in FIELDS:
        got = np.concatenate([p[f] for p in parts], axis=0)
        assert np.array_equal(got, whole[f]), f
    assert all(float(p["slowest"]) == 11.0 for p in parts)          # max over ranks, seen by every rank
    assert int(whole["episodes_done"].sum()) > 0                    # the truncation / auto-reset path ran


def test_partition_arithmetic():
    cfg = dict(n_games=10, game_id_base=5)
    got = [replicas.strong_replica_config(cfg, r, 4) for r in range(4)]
    assert [(c["game_id_base"], c["n_games"]) for c in got] == [(5, 3), (8, 3), (11, 2), (13, 2)]
    assert replicas.weak_replica_config(cfg, 3)["game_id_base"] == 35
    with pytest.raises(ValueError):
        replicas.weak_replica_config(dict(n_games=1 << 31, game_id_base=0), 2)
    assert replicas.max_over_ranks(3.5) == 3.5
