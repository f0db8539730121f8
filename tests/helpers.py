"""Shared test helpers: hand-built boards for the oracle, field lists for parity."""
import numpy as np

STATE_FIELDS = ["army", "owner", "terrain", "turn", "episode", "alive", "general_cell", "land",
                "army_total", "episodes_done", "wins", "truncations", "sat_events", "play_size", "invalid_actions"]
OUT_FIELDS = ["reward", "done", "winner", "obs_army", "obs_owner", "obs_terrain", "obs_vis"]

UP, DOWN, LEFT, RIGHT = 0, 1, 2, 3
PASS = 0


def act(r, c, W, direction, half=0):
    """Flat action index a = cell*9 + 1 + 2*dir + half (R22)."""
    return (r * W + c) * 9 + 1 + 2 * direction + half


def hand_board(oracle_mod, H, W, P, cells, turn=1, team_size=1, **cfg):
    """One game whose state is written by hand.

    cells: {(r, c): (terrain, owner, army)}; everything else is neutral empty plain.
    Generals are found from terrain == GENERAL. Scoreboard and observation are derived by the
    oracle's observe() so that the state is self-consistent before the step under test.
    """
    base = dict(n_games=1, height=H, width=W, n_players=P, team_size=team_size)
    base.update(cfg)
    o = oracle_mod.Oracle(base)
    o.army[:] = 0
    o.owner[:] = -1
    o.terrain[:] = 0
    o.terrain[0, H * W:] = 1
    o.general_cell[:] = -1
    alive = 0
    for (r, c), (t, ow, a) in cells.items():
        i = r * W + c
        o.terrain[0, i], o.owner[0, i], o.army[0, i] = t, ow, a
        if t == oracle_mod.T_GENERAL and ow >= 0 and o.general_cell[0, ow] < 0:   # the first one listed is the general
            o.general_cell[0, ow] = i
            alive |= 1 << ow
    o.alive[0] = alive
    o.turn[0] = turn
    o.winner[:] = -1
    o.observe()
    return o


def cell(o, r, c):
    i = r * o.W + c
    return int(o.terrain[0, i]), int(o.owner[0, i]), int(o.army[0, i])


def snapshot(o, fields):
    return {f: np.array(o.field(f), copy=True) for f in fields}
