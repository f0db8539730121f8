"""An independent replay of the synthetic board generator (SURVEY 8(c) R14 / R30 "exact Philox
replay"; P:L79 is the passage that fixes the map statistics).

The oracle's `generate` was pinned by constraints and marginal statistics only: a biased pick among the candidates,
a swapped Philox word or a wrong counter field would pass those.  Here the generator is written out a second time, in
Python, from the TEXT of DESIGN.md section 3 -- reading R30 (order of the draws, row-major candidate lists, the window
that widens by one on each side while it is empty), R13 / R14 (armies), R29 (Manhattan distance) and the "Philox
streams" table (domain, counter words, which output word serves what) -- on top of a Python Philox4x32-10 that is
itself pinned by the Random123 known answers.  Nothing here reads or calls the oracle's code except to fetch the
boards that are compared, cell for cell.
"""
import numpy as np
import pytest

import workloads

pytestmark = pytest.mark.filterwarnings("ignore")

PLAIN, MOUNTAIN, CITY, GENERAL = 0, 1, 2, 3
DOM_SPAWN, DOM_MOUNTAIN, DOM_CITY = 1, 2, 3


def philox4x32_10(ctr, key):
    """Salmon et al., SC'11: ten rounds of two 32x32 -> 64 multiplies, key bumped by the Weyl constants."""
    c, k = list(ctr), list(key)
    for _ in range(10):
        p0, p1 = 0xD2511F53 * c[0], 0xCD9E8D57 * c[2]
        c = [(p1 >> 32) ^ c[1] ^ k[0], p1 & 0xFFFFFFFF, (p0 >> 32) ^ c[3] ^ k[1], p0 & 0xFFFFFFFF]
        k = [(k[0] + 0x9E3779B9) & 0xFFFFFFFF, (k[1] + 0xBB67AE85) & 0xFFFFFFFF]
    return c


def test_the_replays_philox_matches_the_known_answers():
    """tests/golden/philox_kat.txt (Random123's vectors): the replay below stands on this, not on the oracle."""
    assert philox4x32_10([0] * 4, [0] * 2) == [0x6627e8d5, 0xe169c58d, 0xbc57ac4c, 0x9b00dbd8]
    assert philox4x32_10([0xffffffff] * 4, [0xffffffff] * 2) == [0x408f276d, 0x41c83b0e, 0xa20bc7c6, 0x6d5451fd]
    assert philox4x32_10([0x243f6a88, 0x85a308d3, 0x13198a2e, 0x03707344],
                         [0xa4093822, 0x299f31d0]) == [0xd16cfe09, 0x94fdcceb, 0x5001e420, 0x24126ea1]


def mulhi32(u, n):
    return (u * n) >> 32


def replay(cfg, g, episode=0, trace=None):
    """One board of global game id game_id_base + g, R30's four numbered steps."""
    H, W, P = cfg["height"], cfg["width"], cfg["n_players"]
    HW = H * W
    gid = (cfg.get("game_id_base", 0) + g) & 0xFFFFFFFF
    seed = cfg.get("seed", 0)
    key = (seed & 0xFFFFFFFF, seed >> 32)

    def draw(domain, c0, player=0):
        return philox4x32_10([c0, gid, episode, (domain << 24) | player], key)

    def dist(a, b):
        return abs(a // W - b // W) + abs(a % W - b % W)

    terrain, owner, army = [PLAIN] * HW, [-1] * HW, [0] * HW
    # (1) the spawn window; the curriculum draws the exact distance with word 1 of general 0's call
    lo, hi = cfg["spawn_dmin"], cfg["spawn_dmax"] if cfg["spawn_dmax"] > 0 else 64
    if cfg["spawn_exact"]:
        lo = hi = cfg["spawn_dmin"] + mulhi32(draw(DOM_SPAWN, 0)[1], cfg["spawn_dmax"] - cfg["spawn_dmin"] + 1)
    # (2) generals in player order
    generals = []
    for p in range(P):
        w0 = draw(DOM_SPAWN, p)[0]
        if p == 0:
            cell = mulhi32(w0, HW)
        else:
            l, h = lo, hi
            while True:
                cand = [c for c in range(HW) if c not in generals and l <= min(dist(c, q) for q in generals) <= h]
                if cand:
                    break
                l, h = max(0, l - 1), h + 1
            cell = cand[mulhi32(w0, len(cand))]
            if trace is not None and p == 1:
                trace["general1"] = (cand.index(cell), len(cand))
        generals.append(cell)
        terrain[cell], owner[cell], army[cell] = GENERAL, p, 1                 # R13
    # (3) mountains: one call serves four consecutive cells
    words = {}
    for c in range(HW):
        if terrain[c] == GENERAL:
            continue
        if c >> 2 not in words:
            words[c >> 2] = draw(DOM_MOUNTAIN, c >> 2)
        if words[c >> 2][c & 3] < cfg["mountain_thr"]:
            terrain[c] = MOUNTAIN
    # (4) cities one at a time over what is still plain; garrison from word 1 (R14)
    for k in range(cfg["n_cities"]):
        cand = [c for c in range(HW) if terrain[c] == PLAIN]
        if not cand:
            break
        w = draw(DOM_CITY, k)
        cell = cand[mulhi32(w[0], len(cand))]
        terrain[cell] = CITY
        army[cell] = cfg["city_army_lo"] + mulhi32(w[1], cfg["city_army_hi"] - cfg["city_army_lo"] + 1)
        if trace is not None:
            trace.setdefault("cities", []).append((cand.index(cell), len(cand)))
    return terrain, owner, army, generals


CASES = [
    ("c1_8x8", dict(n_games=40)),
    ("c2_24x24", dict(n_games=24)),
    ("c4_curriculum", dict(n_games=24)),                                        # exact distance d ~ U{3..20}
    ("c5a_2v2", dict(n_games=6)),
    ("c5b_ffa8", dict(n_games=6)),                                              # eight generals, pairwise >= 10
    ("c1_8x8", dict(n_games=24, seed=0x9E3779B97F4A7C15, game_id_base=0xFFFFFF00)),   # 64-bit seed, high game ids
    ("c1_8x8", dict(n_games=24, height=5, width=7, spawn_dmin=9, spawn_dmax=9)),      # a window that must widen
    ("c2_24x24", dict(n_games=12, height=3, width=3, n_cities=9, spawn_dmin=1)),      # more cities than plain cells
]


@pytest.mark.parametrize("name,over", CASES)
def test_generator_replay_cell_for_cell(oracle_mod, name, over):
    cfg, _ = workloads.config(name, **over)
    o = oracle_mod.Oracle(cfg)
    o.reset()
    HW = cfg["height"] * cfg["width"]
    for g in range(cfg["n_games"]):
        terrain, owner, army, generals = replay(cfg, g)
        assert terrain == o.terrain[g, :HW].tolist(), (name, g, "terrain")
        assert owner == o.owner[g, :HW].tolist(), (name, g, "owner")
        assert army == o.army[g, :HW].tolist(), (name, g, "army")
        assert generals == o.general_cell[g].tolist(), (name, g, "general_cell")
        assert (o.terrain[g, HW:] == MOUNTAIN).all() and (o.owner[g, HW:] == -1).all() and (o.army[g, HW:] == 0).all()
    assert (o.turn == 0).all() and (o.alive == (1 << cfg["n_players"]) - 1).all()


def test_generator_replay_of_later_episodes(oracle_mod):
    """The episode counter is counter word c2: the boards an auto-reset generates (R17) replay as well."""
    cfg, _ = workloads.config("c1_8x8", n_games=30, max_turns=6, auto_reset=1)
    o = oracle_mod.Oracle(cfg)
    o.reset()
    for _ in range(6 * 3):                                  # truncation at turn 6: three auto-resets per game
        o.step()
    assert (np.asarray(o.episode) == 3).all() and (o.turn == 0).all()
    for g in range(30):
        terrain, owner, army, generals = replay(cfg, g, episode=3)
        assert terrain == o.terrain[g, :64].tolist() and owner == o.owner[g, :64].tolist(), g
        assert army == o.army[g, :64].tolist() and generals == o.general_cell[g].tolist(), g


def chi2_uniform(us, bins):
    counts = np.bincount(np.minimum((np.asarray(us) * bins).astype(int), bins - 1), minlength=bins)
    e = len(us) / bins
    return float(((counts - e) ** 2 / e).sum())


def test_picks_are_uniform_over_their_candidates(oracle_mod):
    """chi-square of where the oracle's pick falls inside the replay's candidate list (rank / length, 10 bins, 9
    degrees of freedom: 27.9 is the 0.1 % point; the seeds are fixed, so this is a fixed number, not a flaky one):
    general 1 among the cells of its window, every city among the cells still plain."""
    cfg, _ = workloads.config("c2_24x24", n_games=1500, seed=7)
    o = oracle_mod.Oracle(cfg)
    o.reset()
    u_general, u_city = [], []
    for g in range(cfg["n_games"]):
        tr = {}
        terrain, _, _, generals = replay(cfg, g, trace=tr)
        assert terrain == o.terrain[g, :576].tolist() and generals == o.general_cell[g].tolist()
        i, n = tr["general1"]
        u_general.append((i + 0.5) / n)
        u_city += [(i + 0.5) / n for i, n in tr["cities"]]
    assert chi2_uniform(u_general, 10) < 27.9
    assert chi2_uniform(u_city, 10) < 27.9
    # position itself: general 0 is uniform over all 576 cells (24 row bins), cities avoid nothing but non-plain cells
    rows = np.asarray(o.general_cell)[:, 0] // 24
    assert chi2_uniform((rows + 0.5) / 24, 24) < 49.7                          # 23 degrees of freedom, 0.1 % point
