"""Seeded synthetic workloads: the five configs of BASELINE.json as plain dicts.

This module holds NO arithmetic of the method. It only names sizes, thresholds and
seeds, and draws explicit action streams for tests, so that the CUDA path and the CPU
oracle (which share no code) can be fed identical inputs. The recipe follows the
paper's stated map statistics (section IV-A: 20 % mountains, ~10 castles
with 40-50 units, boards up to the 23x23 class) on BASELINE.json's synthetic shapes;
they stand in for the paper's unstated Table I workload.
"""
import numpy as np


def thr(num, den=100):
    """Probability num/den as the uint32 threshold floor(p * 2^32) the library takes."""
    return min((num << 32) // den, 0xFFFFFFFF)


_BASE = dict(team_size=1, city_army_lo=40, city_army_hi=50, spawn_dmax=0, spawn_exact=0,
             max_turns=0, auto_reset=0, rule_flags=0, game_id_base=0, half_thr=thr(50),
             bias_thr=0, seed=0)

# name -> (config dict, steps). n_games is the paper-sized batch; tests shrink it.
CONFIGS = {
    # config 1: 1v1 8x8, 64 games, 300 steps, 15 % mountains, 3 cities, dmin 5, 10 % pass
    "c1_8x8": (dict(_BASE, n_games=64, height=8, width=8, n_players=2, mountain_thr=thr(15),
                    n_cities=3, spawn_dmin=5, pass_thr=thr(10)), 300),
    # config 2: 1v1 24x24, 16,384 games, 2,000 steps, auto-reset, 20 % mountains, 10 cities, dmin 15
    "c2_24x24": (dict(_BASE, n_games=16384, height=24, width=24, n_players=2, mountain_thr=thr(20),
                      n_cities=10, spawn_dmin=15, pass_thr=thr(5), auto_reset=1, max_turns=1000), 2000),
    # config 3: batch sweep on config-2 boards, 1,000 steps (n_games set by the caller)
    "c3_sweep": (dict(_BASE, n_games=262144, height=24, width=24, n_players=2, mountain_thr=thr(20),
                      n_cities=10, spawn_dmin=15, pass_thr=thr(5), auto_reset=1, max_turns=1000), 1000),
    # config 4: spawn-distance curriculum d ~ U{3..20}, 70 % largest-stack bias
    "c4_curriculum": (dict(_BASE, n_games=65536, height=24, width=24, n_players=2, mountain_thr=thr(20),
                           n_cities=10, spawn_dmin=3, spawn_dmax=20, spawn_exact=1, pass_thr=thr(5),
                           bias_thr=thr(70), auto_reset=1, max_turns=2000), 4000),
    # config 5a: 2v2 on 32x32; 5b: 8-player free-for-all
    "c5a_2v2": (dict(_BASE, n_games=32768, height=32, width=32, n_players=4, team_size=2,
                     mountain_thr=thr(20), n_cities=16, spawn_dmin=10, pass_thr=0, auto_reset=1,
                     max_turns=1000), 2000),
    "c5b_ffa8": (dict(_BASE, n_games=32768, height=32, width=32, n_players=8, team_size=1,
                      mountain_thr=thr(20), n_cities=16, spawn_dmin=10, pass_thr=0, auto_reset=1,
                      max_turns=1000), 2000),
    # NEXT-3 (R36): the official generator on the paper's own parameters: up to 23x23, 20 % mountains, 9-11
    # castles of 40-50, generals >= 17 BFS steps apart, a castle within 6 steps of each general, playable area
    # from 18x18 up, padded with mountains
    "official_23x23": (dict(_BASE, n_games=16384, height=23, width=23, n_players=2, mountain_thr=thr(20),
                            n_cities=9, n_cities_max=11, spawn_dmin=17, pass_thr=thr(5), auto_reset=1, max_turns=1000,
                            map_mode=1, play_min=18, castle_radius=6), 2000),
}


def config(name, **overrides):
    cfg, steps = CONFIGS[name]
    cfg = dict(cfg)
    cfg.update(overrides)
    return cfg, steps


def random_actions(rng, n_games, n_players, height, width, p_garbage=0.05):
    """Explicit action stream for tests: uniform over the H*W*9 action space, with a few
    out-of-range values mixed in (they must be treated as passes)."""
    a = rng.integers(0, 9 * height * width, size=(n_games, n_players), dtype=np.int64)
    bad = rng.random((n_games, n_players)) < p_garbage
    junk = rng.choice(np.array([-1, -7, 9 * height * width, 2**31 - 1, -2**31]), size=(n_games, n_players))
    return np.where(bad, junk, a).astype(np.int32)
