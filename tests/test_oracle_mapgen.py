"""Pins of the oracle's official map generator (PAPER.md IV-A P:L79, VI-C P:L169, App. A P:L312;
DESIGN R36).  The paper prints no example map, so the generator is pinned by the constraints the paper states, checked
with an INDEPENDENT shortest-path routine (scipy.sparse.csgraph on the grid graph, not the oracle's queue), by
closed forms on mountain-free boards (steps = Manhattan distance), by tiny boards whose accepted maps can be listed
by hand, and by the statistics of the draws."""
import numpy as np
import pytest
from scipy.sparse import coo_matrix
from scipy.sparse.csgraph import shortest_path

import workloads

PL, MT, CT, GN = 0, 1, 2, 3
OFFICIAL = dict(map_mode=1, height=23, width=23, n_cities=9, n_cities_max=11, spawn_dmin=17, castle_radius=6,
                auto_reset=0, max_turns=0)


def grid_distances(terrain, H, W, src):
    """Steps from src to every cell over non-mountain cells (4-neighbourhood), by scipy's shortest_path."""
    t = terrain[:H * W].reshape(H, W)
    idx = np.arange(H * W).reshape(H, W)
    ok = t != MT
    rows, cols = [], []
    for a, b in ((idx[:, :-1], idx[:, 1:]), (idx[:-1, :], idx[1:, :])):
        m = ok.ravel()[a.ravel()] & ok.ravel()[b.ravel()]
        rows += [a.ravel()[m], b.ravel()[m]]
        cols += [b.ravel()[m], a.ravel()[m]]
    rows, cols = np.concatenate(rows), np.concatenate(cols)
    g = coo_matrix((np.ones(len(rows)), (rows, cols)), shape=(H * W, H * W)).tocsr()
    return shortest_path(g, method="D", unweighted=True, indices=src)


def make(oracle_mod, n_games, **over):
    cfg, _ = workloads.config("c2_24x24", n_games=n_games, **dict(OFFICIAL, **over))
    o = oracle_mod.Oracle(cfg)
    o.reset()
    return o


def test_official_constraints_hold_on_every_map(oracle_mod):
    """P:L79 on the paper's own parameters (23x23, 20 % mountains, 9-11 castles of 40-50, generals >= 17 steps apart,
    a castle within 6 steps of each general), checked with an independent shortest-path routine."""
    N, H, W = 300, 23, 23
    o = make(oracle_mod, N)
    counts = []
    for g in range(N):
        t, ow, a = o.terrain[g], o.owner[g], o.army[g]
        g0, g1 = int(o.general_cell[g, 0]), int(o.general_cell[g, 1])
        assert g0 != g1 and t[g0] == GN and t[g1] == GN and ow[g0] == 0 and ow[g1] == 1 and a[g0] == 1 and a[g1] == 1
        assert (t[:H * W] == GN).sum() == 2
        d0, d1 = grid_distances(t, H, W, g0), grid_distances(t, H, W, g1)
        assert np.isfinite(d0[g1]) and d0[g1] >= 17                     # connected, at least 17 steps apart
        castles = np.flatnonzero(t[:H * W] == CT)
        counts.append(len(castles))
        assert 9 <= len(castles) <= 11
        assert ((a[castles] >= 40) & (a[castles] <= 50)).all() and (ow[castles] == -1).all()
        assert d0[castles].min() <= 6 and d1[castles].min() <= 6         # a castle within radius 6 of each general
        other = np.ones(o.S, bool)
        other[castles] = False
        other[[g0, g1]] = False
        assert (a[other] == 0).all() and (ow[other] == -1).all()
        assert (t[H * W:] == MT).all()                                    # stride padding reads as mountain
    assert int(o.turn.max()) == 0 and (o.alive == 3).all()
    assert set(counts) == {9, 10, 11}
    assert min(np.bincount(counts)[9:]) > N / 3 - 4 * np.sqrt(N * 2 / 9)  # uniform over {9, 10, 11}
    m = (o.terrain[:, :H * W] == MT).mean()
    assert abs(m - 0.2) < 0.01, m                                         # "a random 20 % of cells"


def test_playable_area_is_padded_with_mountains(oracle_mod):
    """cells outside the playable area are mountains; the playable size is uniform in [play_min, H] x [.., W]."""
    N, H, W = 400, 23, 23
    o = make(oracle_mod, N, play_min=18)
    hs, ws = [], []
    for g in range(N):
        t = o.terrain[g, :H * W].reshape(H, W)
        free = t != MT
        r = np.flatnonzero(free.any(1)).max() + 1
        c = np.flatnonzero(free.any(0)).max() + 1
        hs.append(r)
        ws.append(c)
        assert (t[r:, :] == MT).all() and (t[:, c:] == MT).all()
    assert min(hs) >= 18 and min(ws) >= 18 and max(hs) == 23 and max(ws) == 23
    # the last free row is the playable height unless that whole row drew mountains (0.2^18: never in 400 games)
    for vals in (hs, ws):
        cnt = np.bincount(vals, minlength=24)[18:]
        assert cnt.min() > N / 6 - 4 * np.sqrt(N * 5 / 36), cnt


def test_mountain_free_board_is_manhattan(oracle_mod):
    """Closed form: without mountains the step distance is the Manhattan distance, so with spawn_exact the generals sit
    at exactly the drawn d, d uniform over {3..20} (the curriculum of P:L169), and castles 0 / 1 lie within Manhattan
    radius 6 of generals 0 / 1 -- no path-finding involved in the check."""
    N, H, W = 2000, 23, 23
    o = make(oracle_mod, N, mountain_thr=0, spawn_dmin=3, spawn_dmax=20, spawn_exact=1)
    g = o.general_cell.astype(int)
    d = np.abs(g[:, 0] // W - g[:, 1] // W) + np.abs(g[:, 0] % W - g[:, 1] % W)
    assert d.min() == 3 and d.max() == 20
    cnt = np.bincount(d, minlength=21)[3:]
    assert cnt.min() > N / 18 - 4 * np.sqrt(N / 18), cnt
    for k in range(N):
        cells = np.flatnonzero(o.terrain[k, :H * W] == CT)
        for p in range(2):
            dm = np.abs(cells // W - g[k, p] // W) + np.abs(cells % W - g[k, p] % W)
            assert dm.min() <= 6


def test_tiny_boards_by_hand(oracle_mod):
    """1 x 5 without mountains, generals at least 4 steps apart: the only accepted maps put them on the two end
    cells (a first general anywhere else leaves no cell 4 steps away and the attempt is rejected); both orders occur.
    One castle, radius 1: it sits next to general 0."""
    N = 600
    cfg, _ = workloads.config("c2_24x24", n_games=N, map_mode=1, height=1, width=5, mountain_thr=0, n_cities=1,
                              n_cities_max=0, spawn_dmin=4, castle_radius=1, auto_reset=0)
    o = oracle_mod.Oracle(cfg)
    o.reset()
    g = o.general_cell.astype(int)
    assert set(map(tuple, g)) == {(0, 4), (4, 0)}
    assert abs((g[:, 0] == 0).mean() - 0.5) < 4 * 0.5 / np.sqrt(N)
    for k in range(N):
        castle = np.flatnonzero(o.terrain[k, :5] == CT)
        assert len(castle) == 1 and abs(castle[0] - g[k, 0]) == 1


def test_second_general_is_uniform_over_the_qualifying_cells(oracle_mod):
    """4 x 4 without mountains, at least 5 steps apart, no castles.  By hand: a corner has 3 cells at >= 5 steps (the
    opposite corner and its two neighbours), an edge cell (x, 0) with x in {1, 2} has exactly one (the far corner of
    the opposite side), an inner cell none.  So of the accepted maps those with general 0 in a corner are
    4 x 3 / (4 x 3 + 8 x 1) ... but acceptance is per attempt, not per cell: an attempt is accepted iff general 0 is
    not an inner cell (12 / 16), each non-inner cell equally likely => P(corner) = 4 / 12; given a corner, general 1 is
    uniform over its three cells."""
    N, H, W = 3000, 4, 4
    cfg, _ = workloads.config("c2_24x24", n_games=N, map_mode=1, height=H, width=W, mountain_thr=0, n_cities=0,
                              spawn_dmin=5, castle_radius=0, auto_reset=0)
    o = oracle_mod.Oracle(cfg)
    o.reset()
    g = o.general_cell.astype(int)
    d = np.abs(g[:, 0] // W - g[:, 1] // W) + np.abs(g[:, 0] % W - g[:, 1] % W)
    assert d.min() >= 5
    corners = {0, 3, 12, 15}
    inner = {5, 6, 9, 10}
    assert not (set(g[:, 0]) & inner)
    is_corner = np.isin(g[:, 0], list(corners))
    assert abs(is_corner.mean() - 1 / 3) < 4 * np.sqrt(2 / 9 / N)
    sel = g[g[:, 0] == 0, 1]
    assert set(sel) == {15, 14, 11}
    cnt = np.bincount(sel, minlength=16)[[15, 14, 11]]
    assert cnt.min() > len(sel) / 3 - 4 * np.sqrt(len(sel) * 2 / 9)


def test_maps_are_a_function_of_seed_game_and_episode(oracle_mod):
    """M2 for the official generator: a game depends on its global id only; a new episode draws a new map."""
    a = make(oracle_mod, 12)
    b = make(oracle_mod, 5, game_id_base=7)
    assert np.array_equal(a.terrain[7:12], b.terrain) and np.array_equal(a.army[7:12], b.army)
    assert np.array_equal(a.general_cell[7:12], b.general_cell)
    c = make(oracle_mod, 12, seed=1)
    assert not np.array_equal(a.terrain, c.terrain)
    # auto-reset regenerates with episode + 1: play short truncated episodes and compare with a fresh episode-1 map
    o = make(oracle_mod, 6, auto_reset=1, max_turns=3, spawn_dmin=17)
    first = o.terrain.copy()
    for _ in range(3):
        o.step()
    assert (o.episode == 1).all() and (o.turn == 0).all()
    assert not np.array_equal(first, o.terrain)
    for g in range(6):
        t = o.terrain[g]
        g0, g1 = int(o.general_cell[g, 0]), int(o.general_cell[g, 1])
        assert grid_distances(t, 23, 23, g0)[g1] >= 17


def test_play_on_official_maps_keeps_the_invariants(oracle_mod):
    """The step rules do not care which generator made the board: ownership / terrain consistency and the public
    scoreboard stay exact over sampled play with auto-reset."""
    o = make(oracle_mod, 24, auto_reset=1, max_turns=120, spawn_dmin=4, spawn_dmax=8, pass_thr=workloads.thr(5))
    for _ in range(400):
        o.step()
        HW = 23 * 23
        owner, army, terrain = o.owner[:, :HW], o.army[:, :HW], o.terrain[:, :HW]
        assert (owner[terrain == MT] == -1).all() and (army >= 0).all()
        for p in range(2):
            assert np.array_equal(o.land[:, p], (owner == p).sum(1))
            assert np.array_equal(o.army_total[:, p], (army.astype(np.int64) * (owner == p)).sum(1))
    assert int(o.episodes_done.sum()) > 24
