"""Pins for the CPU oracle beyond the hand-worked examples: closed forms C1..C3, invariants I1..I7,
brute force B1/B2, metamorphic M1/M2, generator statistics, auto-reset convention (R17) and the
digest definition (R28).  Nothing here calls the CUDA path; expected values come from the rules of
PAPER.md section IV restated independently in Python, or from closed forms.
"""
import numpy as np
import pytest

from helpers import DOWN, LEFT, PASS, RIGHT, UP, act, cell, hand_board
import workloads

PL, MT, CT, GN = 0, 1, 2, 3
M64 = (1 << 64) - 1


# --------------------------------------------------------------------------- closed forms
@pytest.mark.parametrize("flags,T", [(0, 120), (1, 120)])
def test_C1_all_pass_growth_closed_form(oracle_mod, flags, T):
    """P:L87 + R1/R2: general = 1 + floor(T/2) + floor(T/50) (TICK_PLAIN_ONLY: 1 + floor(T/2))."""
    cfg, _ = workloads.config("c1_8x8", n_games=8, rule_flags=flags)
    o = oracle_mod.Oracle(cfg)
    o.reset()
    terrain0, owner0 = o.terrain.copy(), o.owner.copy()
    army0 = o.army.copy()
    for t in range(1, T + 1):
        o.step(np.zeros((8, 2), np.int32))
        want = 1 + t // 2 + (0 if flags else t // 50)
        for g in range(8):
            for p in range(2):
                gc = int(o.general_cell[g, p])
                assert int(o.army[g, gc]) == want
        assert (o.land == 1).all() and (o.army_total == want).all()
        assert (o.turn == t).all() and (o.done[0] == 0).all()
    assert np.array_equal(o.terrain, terrain0) and np.array_equal(o.owner, owner0)
    changed = o.army != army0
    assert changed.sum() == 16            # only the 2 generals of each of the 8 games


@pytest.mark.parametrize("r,c,want", [(0, 0, 4), (0, 3, 6), (3, 3, 9), (6, 6, 4), (6, 2, 6), (2, 0, 6)])
def test_C2_lone_cell_visibility_count(oracle_mod, r, c, want):
    """a player sees its cells and their 8 neighbours, clipped at the border."""
    H = W = 7
    cells = {(r, c): (GN, 0, 1)}
    far = (0, 6) if (r, c) != (0, 6) and abs(r - 0) + abs(c - 6) > 3 else (6, 0)
    cells[far] = (GN, 1, 1)
    o = hand_board(oracle_mod, H, W, 2, cells)
    vis = o.obs_vis[0, 0, 0, :H * W].reshape(H, W)
    assert int(vis.sum()) == want
    rr, cc = np.nonzero(vis)
    assert rr.min() == max(r - 1, 0) and rr.max() == min(r + 1, H - 1)
    assert cc.min() == max(c - 1, 0) and cc.max() == min(c + 1, W - 1)


def test_C3_growth_counts_between_turns(oracle_mod):
    """plain +1 per multiple of 50 in (t0, t0+T]; castle/general additionally +1 per even turn."""
    t0, T = 37, 130
    cells = {(0, 0): (GN, 0, 1), (4, 4): (GN, 1, 1), (0, 2): (PL, 0, 7), (2, 2): (CT, 0, 3),
             (3, 0): (CT, -1, 44), (4, 0): (PL, -1, 0), (1, 4): (PL, 1, 9)}
    o = hand_board(oracle_mod, 5, 5, 2, cells, turn=t0)
    for _ in range(T):
        o.step([[PASS, PASS]])
    n50 = (t0 + T) // 50 - t0 // 50
    n2 = (t0 + T) // 2 - t0 // 2
    assert cell(o, 0, 2) == (PL, 0, 7 + n50)
    assert cell(o, 1, 4) == (PL, 1, 9 + n50)
    assert cell(o, 2, 2) == (CT, 0, 3 + n50 + n2)
    assert cell(o, 0, 0) == (GN, 0, 1 + n50 + n2)
    assert cell(o, 3, 0) == (CT, -1, 44)          # neutral castles never grow
    assert cell(o, 4, 0) == (PL, -1, 0)


# --------------------------------------------------------------------------- independent restatement
def py_valid(army, owner, terrain, H, W, p, a):
    """Validity predicate of a2 restated from P:L79 (mountain impassable), P:L91 (owned source,
    all-but-one / half => at least 2 units), R10 (no wrap-around)."""
    if a < 0 or a >= 9 * H * W:
        return None
    c, k = divmod(a, 9)
    if k == 0:
        return None
    d, half = divmod(k - 1, 2)
    r, col = divmod(c, W)
    r2, c2 = r + (-1, 1, 0, 0)[d], col + (0, 0, -1, 1)[d]
    if not (0 <= r2 < H and 0 <= c2 < W):
        return None
    t = r2 * W + c2
    if owner[c] != p or army[c] < 2 or terrain[t] == MT:
        return None
    return c, t, half


def py_philox(ctr, key):
    """Philox4x32-10 restated (pinned by the Random123 vectors in test_oracle_pins)."""
    c, k = list(ctr), list(key)
    for _ in range(10):
        p0, p1 = 0xD2511F53 * c[0], 0xCD9E8D57 * c[2]
        c = [(p1 >> 32) ^ c[1] ^ k[0], p1 & 0xFFFFFFFF, (p0 >> 32) ^ c[3] ^ k[1], p0 & 0xFFFFFFFF]
        k = [(k[0] + 0x9E3779B9) & 0xFFFFFFFF, (k[1] + 0xBB67AE85) & 0xFFFFFFFF]
    return c


def test_py_philox_matches_kat():
    assert py_philox([0] * 4, [0] * 2) == [0x6627e8d5, 0xe169c58d, 0xbc57ac4c, 0x9b00dbd8]
    assert py_philox([0x243f6a88, 0x85a308d3, 0x13198a2e, 0x03707344],
                     [0xa4093822, 0x299f31d0]) == [0xd16cfe09, 0x94fdcceb, 0x5001e420, 0x24126ea1]


def _random_small_board(oracle_mod, rng, H, W, P=2, team_size=1, **cfg):
    cells = {}
    free = [(r, c) for r in range(H) for c in range(W)]
    rng.shuffle(free)
    for p in range(P):
        cells[free.pop()] = (GN, p, int(rng.integers(1, 6)))
    for rc in free:
        u = rng.random()
        if u < 0.15:
            cells[rc] = (MT, -1, 0)
        elif u < 0.25:
            cells[rc] = (CT, int(rng.integers(-1, P)), int(rng.integers(0, 8)))
        elif u < 0.7:
            ow = int(rng.integers(-1, P))
            cells[rc] = (PL, ow, int(rng.integers(0, 7)) if ow >= 0 else 0)
    return hand_board(oracle_mod, H, W, P, cells, turn=int(rng.integers(0, 5)) * 2, team_size=team_size,
                      **cfg)


def _clone_state(o, oracle_mod):
    d = {k: getattr(o.cfg, k) for k in ("n_games", "height", "width", "n_players", "team_size",
                                        "max_turns", "auto_reset", "rule_flags", "pass_thr", "half_thr",
                                        "bias_thr", "seed", "game_id_base")}
    n = oracle_mod.Oracle(d)
    for f in ("army", "owner", "terrain", "turn", "episode", "alive", "general_cell", "land",
              "army_total", "done", "winner"):
        getattr(n, f)[...] = getattr(o, f)
    return n


@pytest.mark.parametrize("H,W", [(2, 3), (3, 3), (4, 4)])
def test_B1_every_action_changes_board_iff_valid(oracle_mod, H, W):
    """I6 / B1: enumerate all 9*H*W actions (plus out-of-range ones) for each player: the board
    changes (beyond growth) iff the restated predicate holds, and then exactly as P:L91-93 says."""
    rng = np.random.default_rng(H * 10 + W)
    for _ in range(12):
        base = _random_small_board(oracle_mod, rng, H, W)
        ref = _clone_state(base, oracle_mod)
        ref.step([[PASS, PASS]])
        for p in range(2):
            for a in list(range(-2, 9 * H * W + 3)):
                o = _clone_state(base, oracle_mod)
                acts = [PASS, PASS]
                acts[p] = a
                o.step([acts])
                v = py_valid(base.army[0], base.owner[0], base.terrain[0], H, W, p, a)
                same = np.array_equal(o.army, ref.army) and np.array_equal(o.owner, ref.owner)
                if v is None:
                    assert same, (p, a)
                    continue
                src, dst, half = v
                a_src = int(base.army[0, src])
                m = a_src // 2 if half else a_src - 1
                grow = lambda c, st: int(st.army[0, c]) - 0    # noqa: E731
                # undo growth: compare against the pass-run's growth on untouched cells
                assert not same or m == 0, (p, a)
                d, t = int(base.army[0, dst]), int(base.owner[0, dst])
                if t == p:
                    want_owner, want = p, d + m
                elif m > d:
                    want_owner, want = p, m - d
                else:
                    want_owner, want = t, d - m
                was_general = int(base.terrain[0, dst]) == GN and t != p and m > d
                g_src = int(ref.army[0, src]) - a_src                     # growth the pass-run gave
                assert int(o.army[0, src]) == a_src - m + g_src
                assert int(o.owner[0, dst]) == want_owner
                if not was_general:
                    g_dst = 0
                    if want_owner >= 0 and int(o.turn[0]) % 2 == 0 and int(base.terrain[0, dst]) in (CT, GN):
                        g_dst = 1
                    assert int(o.army[0, dst]) == want + g_dst, (p, a)
                    # nothing else moved
                    mask = np.ones(H * W, bool)
                    mask[[src, dst]] = False
                    assert np.array_equal(o.army[0, :H * W][mask], ref.army[0, :H * W][mask])
                    assert np.array_equal(o.owner[0, :H * W][mask], ref.owner[0, :H * W][mask])
                else:
                    assert int(o.terrain[0, dst]) == CT and int(o.done[0, 0]) == 1
                    assert (o.owner[0, :H * W] != t).all()


@pytest.mark.parametrize("bias", [0, 70])
def test_B2_sampler_follows_its_definition(oracle_mod, bias):
    """R24/R25: pass iff w0 < pass_thr; otherwise the mulhi32(w1, n)-th entry of the valid list in
    (direction, cell) order (restricted to the largest owned stack iff w3 < bias_thr and that stack
    can move); half iff w2 < half_thr.  Valid list == board-changing 'all' moves (brute force)."""
    rng = np.random.default_rng(7 + bias)
    H, W = 4, 5
    seed = 0x1234567890ABCDEF
    n_pass = n_move = 0
    for trial in range(40):
        base = _random_small_board(oracle_mod, rng, H, W, seed=seed, pass_thr=workloads.thr(10),
                                   half_thr=workloads.thr(50), bias_thr=workloads.thr(bias),
                                   game_id_base=1000 + trial)
        army, owner, terrain = base.army[0], base.owner[0], base.terrain[0]
        for step in range(6):
            base.global_step = step
            got = base.sample()[0]
            for p in range(2):
                w = py_philox([0, 1000 + trial, step, (4 << 24) | p], [seed & 0xFFFFFFFF, seed >> 32])
                valid = [c * 9 + 1 + 2 * d for d in range(4) for c in range(H * W)
                         if py_valid(army, owner, terrain, H, W, p, c * 9 + 1 + 2 * d)]
                if w[0] < workloads.thr(10) or not valid:
                    assert got[p] == 0
                    n_pass += 1
                    continue
                if w[3] < workloads.thr(bias):
                    owned = [c for c in range(H * W) if owner[c] == p]
                    best = max(owned, key=lambda c: (int(army[c]), -c))
                    sub = [a for a in valid if a // 9 == best]
                    if sub:
                        valid = sub
                want = valid[(w[1] * len(valid)) >> 32] + (1 if w[2] < workloads.thr(50) else 0)
                assert got[p] == want
                n_move += 1
    assert n_pass > 10 and n_move > 100


def test_B2_sampler_uniform_over_valid_moves(oracle_mod):
    """chi-square: over many (game id, step) draws on one fixed board every valid move is equally likely."""
    cells = {(0, 0): (GN, 0, 5), (0, 1): (PL, 0, 3), (1, 0): (PL, 0, 2), (1, 1): (MT, -1, 0),
             (3, 3): (GN, 1, 1), (2, 0): (PL, 0, 1)}
    counts = {}
    n = 0
    for gid in range(60):
        o = hand_board(oracle_mod, 4, 4, 2, cells, pass_thr=0, half_thr=workloads.thr(50),
                       seed=99, game_id_base=gid)
        for step in range(100):
            o.global_step = step
            a = int(o.sample()[0, 0])
            counts[a] = counts.get(a, 0) + 1
            n += 1
    # valid 'all' moves of P0: (0,0) down/right, (0,1) left/right (down is mountain), (1,0) up/down
    # -> 6 moves x {all, half} = 12 actions
    assert len(counts) == 12
    exp = n / 12
    chi2 = sum((v - exp) ** 2 / exp for v in counts.values())
    assert chi2 < 40.0                     # 11 dof: P(chi2 > 40) < 4e-5


# --------------------------------------------------------------------------- invariants on random play
def _check_invariants(o, oracle_mod, g_prev):
    H, W, P, HW = o.H, o.W, o.P, o.HW
    for g in range(o.N):
        army, owner, terrain = o.army[g, :HW], o.owner[g, :HW], o.terrain[g, :HW]
        # I2 terrain / owner consistency
        mt = terrain == MT
        assert (owner[mt] == -1).all() and (army[mt] == 0).all()
        assert (army >= 0).all()
        alive = int(o.alive[g])
        assert int((terrain == GN).sum()) == bin(alive).count("1")
        for p in range(P):
            gc = int(o.general_cell[g, p])
            if (alive >> p) & 1:
                assert terrain[gc] == GN and owner[gc] == p
            else:
                assert gc == -1
                assert not (owner == p).any()              # I3: eliminated players own nothing
        # I4 scoreboard equals a recount
        for p in range(P):
            assert int(o.land[g, p]) == int((owner == p).sum())
            assert int(o.army_total[g, p]) == int(army[owner == p].astype(np.int64).sum())
        # I5 fog
        team = lambda q: q // max(1, o.cfg.team_size)      # noqa: E731
        for p in range(P):
            mine = np.isin(owner, [q for q in range(P) if team(q) == team(p)]).reshape(H, W)
            pad = np.pad(mine, 1)
            vis = np.zeros((H, W), bool)
            for dr in range(3):
                for dc in range(3):
                    vis |= pad[dr:dr + H, dc:dc + W]
            vis = vis.reshape(-1)
            assert np.array_equal(o.obs_vis[0, g, p, :HW].astype(bool), vis)
            assert np.array_equal(o.obs_army[0, g, p, :HW], np.where(vis, army, 0))
            assert np.array_equal(o.obs_owner[0, g, p, :HW], np.where(vis, owner, -2))
            assert np.array_equal(o.obs_terrain[0, g, p, :HW], np.where(vis, terrain, 4))
        # I7 rewards
        rs = o.reward[0, g].astype(int)
        if g_prev is not None and g_prev[g] and not o.cfg.auto_reset:
            assert (rs == 0).all()                         # R31: frozen game, reward 0, done kept
        elif int(o.done[0, g]) & 1:
            assert sorted(set(rs.tolist())) == [-1, 1]
            assert int(o.winner[0, g]) >= 0
        else:
            assert (rs == 0).all() and int(o.winner[0, g]) == -1


@pytest.mark.parametrize("name,N,T,over", [
    ("c1_8x8", 16, 300, {}),
    ("c4_curriculum", 6, 400, dict(height=10, width=12, spawn_dmax=9, n_cities=4)),
    ("c5a_2v2", 4, 300, dict(height=9, width=9, spawn_dmin=4, n_cities=3, max_turns=250)),
    ("c5b_ffa8", 3, 300, dict(height=10, width=10, spawn_dmin=3, n_cities=3, max_turns=250)),
])
def test_invariants_on_sampled_play(oracle_mod, name, N, T, over):
    cfg, _ = workloads.config(name, n_games=N, **over)
    o = oracle_mod.Oracle(cfg)
    o.reset()
    _check_invariants(o, oracle_mod, None)
    ended = 0
    for t in range(T):
        prev = o.done[0].copy()
        o.step()
        _check_invariants(o, oracle_mod, prev)
        ended += int(((o.done[0] != 0) & ((prev == 0) | bool(cfg["auto_reset"]))).sum())
    assert (o.sat_events == 0).all()
    if cfg["auto_reset"]:
        assert ended > 0 and int(o.episodes_done.sum()) == ended


def test_I1_army_conservation(oracle_mod):
    """I1: the total army changes only by -2*min(m, d) per hostile move, the halving on capture,
    and growth (one per owned structure on even turns, one per owned cell on multiples of 50)."""
    rng = np.random.default_rng(3)
    H = W = 6
    for trial in range(30):
        o = _random_small_board(oracle_mod, rng, H, W)
        for _ in range(20):
            if int(o.done[0, 0]):
                break
            army, owner, terrain = o.army[0].copy(), o.owner[0].copy(), o.terrain[0].copy()
            acts = workloads.random_actions(rng, 1, 2, H, W)
            # boost the share of valid moves
            for p in range(2):
                cand = [a for a in range(9 * H * W) if py_valid(army, owner, terrain, H, W, p, a)]
                if cand and rng.random() < 0.8:
                    acts[0, p] = cand[int(rng.integers(len(cand)))]
            total = int(army[:H * W].astype(np.int64)[owner[:H * W] >= 0].sum())
            neutral = int(army[:H * W].astype(np.int64)[owner[:H * W] < 0].sum())
            a2, o2, t2 = army.copy().astype(np.int64), owner.copy(), terrain.copy()
            loss = 0
            for p in range(2):
                v = py_valid(a2, o2, t2, H, W, p, int(acts[0, p]))
                if v is None:
                    continue
                src, dst, half = v
                m = int(a2[src]) // 2 if half else int(a2[src]) - 1
                a2[src] -= m
                d, t = int(a2[dst]), int(o2[dst])
                if t == p:
                    a2[dst] += m
                elif m > d:
                    a2[dst], o2[dst] = m - d, p
                    loss += 2 * d
                    if t2[dst] == GN:
                        t2[dst] = CT
                        for c in range(H * W):
                            if o2[c] == t:
                                loss += int(a2[c]) // 2
                                a2[c] = (a2[c] + 1) // 2
                                o2[c] = p
                else:
                    a2[dst] = d - m
                    loss += 2 * m
            o.step(acts)
            turn = int(o.turn[0])
            owned = o2[:H * W] >= 0
            grow = 0
            if turn % 2 == 0:
                grow += int((owned & np.isin(t2[:H * W], [CT, GN])).sum())
            if turn % 50 == 0:
                grow += int(owned.sum())
            after = int(o.army[0, :H * W].astype(np.int64).sum())
            assert after == total + neutral - loss + grow


# --------------------------------------------------------------------------- metamorphic
def test_M1_reflection_commutes_with_step(oracle_mod):
    """Mirror the board left-right and swap LEFT/RIGHT in the actions: the result is the mirror image."""
    rng = np.random.default_rng(11)
    H, W = 5, 6
    for _ in range(25):
        o = _random_small_board(oracle_mod, rng, H, W)
        m = _clone_state(o, oracle_mod)
        for f in ("army", "owner", "terrain"):
            getattr(m, f)[0, :H * W] = getattr(o, f)[0, :H * W].reshape(H, W)[:, ::-1].reshape(-1)
        for p in range(2):
            gc = int(o.general_cell[0, p])
            m.general_cell[0, p] = (gc // W) * W + (W - 1 - gc % W) if gc >= 0 else -1
        m.observe()
        for _ in range(6):
            acts = workloads.random_actions(rng, 1, 2, H, W, p_garbage=0.0)
            macts = acts.copy()
            for p in range(2):
                c, k = divmod(int(acts[0, p]), 9)
                mc = (c // W) * W + (W - 1 - c % W)
                if k:
                    d, half = divmod(k - 1, 2)
                    d = {LEFT: RIGHT, RIGHT: LEFT}.get(d, d)
                    k = 1 + 2 * d + half
                macts[0, p] = mc * 9 + k
            o.step(acts)
            m.step(macts)
            for f in ("army", "owner", "terrain"):
                a = getattr(o, f)[0, :H * W].reshape(H, W)[:, ::-1].reshape(-1)
                assert np.array_equal(a, getattr(m, f)[0, :H * W])
            assert np.array_equal(o.reward, m.reward) and np.array_equal(o.done, m.done)
            assert np.array_equal(o.obs_vis[0, 0, :, :H * W].reshape(2, H, W)[:, :, ::-1],
                                  m.obs_vis[0, 0, :, :H * W].reshape(2, H, W))


def test_M2_batch_independence_and_rollout_equals_steps(oracle_mod):
    """A game's trajectory depends on (seed, global game id) only: not on N, not on game_id_base
    splits, not on step-by-step vs rollout(K)."""
    cfg, _ = workloads.config("c1_8x8", n_games=12, auto_reset=1, max_turns=60)
    a = oracle_mod.Oracle(cfg)
    a.reset()
    a.rollout(150)
    parts = []
    for base, n in ((0, 5), (5, 7)):
        cfg2, _ = workloads.config("c1_8x8", n_games=n, game_id_base=base, auto_reset=1, max_turns=60)
        b = oracle_mod.Oracle(cfg2)
        b.reset()
        for _ in range(150):
            b.step()
        parts.append(b)
    for f in ("army", "owner", "terrain", "turn", "episode", "land", "army_total", "episodes_done",
              "wins", "obs_digest", "obs_army", "obs_vis", "reward", "done"):
        got = np.concatenate([np.asarray(p.field(f)) for p in parts], axis=0)
        assert np.array_equal(np.asarray(a.field(f)), got), f
    assert int(a.episodes_done.sum()) >= 12


def test_rollout_every_step_slots(oracle_mod):
    cfg, _ = workloads.config("c1_8x8", n_games=6)
    K = 9
    a = oracle_mod.Oracle(cfg, every_step_K=K)
    a.reset()
    a.rollout(K, oracle_mod.OBS_EVERY_STEP)
    b = oracle_mod.Oracle(cfg)
    b.reset()
    for k in range(K):
        b.step()
        assert np.array_equal(a.obs_army[k], b.obs_army[0])
        assert np.array_equal(a.obs_owner[k], b.obs_owner[0])
        assert np.array_equal(a.reward[k], b.reward[0]) and np.array_equal(a.done[k], b.done[0])
    assert np.array_equal(a.obs_digest, b.obs_digest)


# --------------------------------------------------------------------------- auto-reset (R17)
def test_R17_auto_reset_convention(oracle_mod):
    """Up to and including the first done of a game the auto-reset and frozen runs agree on
    reward/done/winner; after it, the auto-reset state equals a fresh generate(seed, gid, episode+1)."""
    cfg_on, _ = workloads.config("c1_8x8", n_games=10, auto_reset=1, max_turns=40)
    cfg_off, _ = workloads.config("c1_8x8", n_games=10, auto_reset=0, max_turns=40)
    on, off = oracle_mod.Oracle(cfg_on), oracle_mod.Oracle(cfg_off)
    on.reset()
    off.reset()
    # fresh boards of episode 1
    fresh = oracle_mod.Oracle(cfg_on)
    fresh.reset()
    seen = np.zeros(10, bool)
    for t in range(45):
        on.step()
        off.step()
        live = ~seen
        assert np.array_equal(on.reward[0][live], off.reward[0][live])
        assert np.array_equal(on.done[0][live], off.done[0][live])
        newly = live & (on.done[0] != 0)
        for g in np.nonzero(newly)[0]:
            assert int(on.episode[g]) == 1 and int(on.turn[g]) == 0
            assert int(on.army[g, on.general_cell[g, 0]]) == 1
            assert int(on.land[g].sum()) == 2
            # frozen copy keeps the terminal board
            assert int(off.turn[g]) == 40
        still = live & ~newly
        assert np.array_equal(on.army[still], off.army[still])
        seen |= newly
    assert seen.all()
    # episode-1 boards differ from episode-0 boards (different Philox counters)
    assert not np.array_equal(on.terrain, fresh.terrain)


# --------------------------------------------------------------------------- generator (a1, R13/R14/R29/R30)
def test_generator_constraints_and_statistics(oracle_mod):
    cfg, _ = workloads.config("c2_24x24", n_games=400)
    o = oracle_mod.Oracle(cfg)
    o.reset()
    HW, W = 576, 24
    mt = 0
    for g in range(400):
        terrain, owner, army = o.terrain[g, :HW], o.owner[g, :HW], o.army[g, :HW]
        g0, g1 = int(o.general_cell[g, 0]), int(o.general_cell[g, 1])
        assert abs(g0 // W - g1 // W) + abs(g0 % W - g1 % W) >= 15          # [B] config 2
        assert terrain[g0] == GN and terrain[g1] == GN and owner[g0] == 0 and owner[g1] == 1
        assert army[g0] == 1 and army[g1] == 1                                 # R13
        assert int((terrain == GN).sum()) == 2
        cities = terrain == CT
        assert int(cities.sum()) == 10                                         # R14
        assert (army[cities] >= 40).all() and (army[cities] <= 50).all()
        assert (owner[cities] == -1).all()
        rest = ~cities
        rest[[g0, g1]] = False
        assert (army[rest] == 0).all() and (owner[rest] == -1).all()
        mt += int((terrain == MT).sum())
    dens = mt / (400 * (HW - 2))
    # Bernoulli(0.2) per non-general cell, then 10 mountains-free picks do not touch mountains
    sigma = (0.2 * 0.8 / (400 * (HW - 2))) ** 0.5
    assert abs(dens - 0.2) < 4 * sigma
    city_armies = o.army[:, :HW][o.terrain[:, :HW] == CT]
    hist = np.bincount(city_armies, minlength=51)[40:51]
    exp = hist.sum() / 11
    assert ((hist - exp) ** 2 / exp).sum() < 35.0          # 10 dof
    # general 0 is uniform over the board: mean row / col near the centre
    rows = o.general_cell[:, 0] // W
    assert abs(rows.mean() - 11.5) < 4 * (47.9 / 400) ** 0.5


def test_generator_exact_spawn_distance(oracle_mod):
    cfg, _ = workloads.config("c4_curriculum", n_games=600)
    o = oracle_mod.Oracle(cfg)
    o.reset()
    W = 24
    g0, g1 = o.general_cell[:, 0].astype(int), o.general_cell[:, 1].astype(int)
    d = np.abs(g0 // W - g1 // W) + np.abs(g0 % W - g1 % W)
    assert d.min() >= 3 and d.max() <= 20
    hist = np.bincount(d, minlength=21)[3:21]
    exp = 600 / 18
    assert (hist > 0).all() and ((hist - exp) ** 2 / exp).sum() < 50.0        # 17 dof


def test_generator_many_players_pairwise_distance(oracle_mod):
    cfg, _ = workloads.config("c5b_ffa8", n_games=50)
    o = oracle_mod.Oracle(cfg)
    o.reset()
    W = 32
    for g in range(50):
        gc = o.general_cell[g].astype(int)
        assert len(set(gc.tolist())) == 8
        for i in range(8):
            for j in range(i):
                assert abs(gc[i] // W - gc[j] // W) + abs(gc[i] % W - gc[j] % W) >= 10
        assert int((o.terrain[g] == CT).sum()) == 16


def test_generator_is_keyed_by_seed_game_episode(oracle_mod):
    cfg, _ = workloads.config("c1_8x8", n_games=4)
    a = oracle_mod.Oracle(cfg)
    a.reset()
    b = oracle_mod.Oracle(dict(cfg, seed=1))
    b.reset()
    c = oracle_mod.Oracle(dict(cfg, game_id_base=2, n_games=2))
    c.reset()
    assert not np.array_equal(a.terrain, b.terrain)
    assert np.array_equal(a.terrain[2:], c.terrain) and np.array_equal(a.army[2:], c.army)
    assert not np.array_equal(a.terrain[0], a.terrain[1])


# --------------------------------------------------------------------------- digest (R28)
def test_digest_definition(oracle_mod):
    """R28 restated with Python integers: per player h = sum_c pack(c) * key(c) mod 2^64 chained by
    mix64, then the step's done / winner / reward bits."""
    def mix(z):
        z &= M64
        z ^= z >> 30
        z = (z * 0xBF58476D1CE4E5B9) & M64
        z ^= z >> 27
        z = (z * 0x94D049BB133111EB) & M64
        return z ^ (z >> 31)

    def key(c):
        return mix(((c + 1) * 0x9E3779B97F4A7C15) & M64) | 1

    cfg, _ = workloads.config("c1_8x8", n_games=3)
    o = oracle_mod.Oracle(cfg)
    o.reset()
    d = [0, 0, 0]

    def chain(d):
        out = []
        for g in range(3):
            x = d[g]
            for p in range(2):
                h = 0
                for c in range(64):
                    pack = (int(o.obs_army[0, g, p, c]) & 0xFFFF) | ((int(o.obs_owner[0, g, p, c]) + 2) << 16) \
                        | (int(o.obs_terrain[0, g, p, c]) << 20) | (int(o.obs_vis[0, g, p, c]) << 24)
                    h = (h + pack * key(c)) & M64
                x = mix(x ^ h)
            tail = int(o.done[0, g]) | (((int(o.winner[0, g]) + 2) & 0xFF) << 8)
            for p in range(2):
                tail |= (int(o.reward[0, g, p]) + 1) << (16 + 2 * p)
            out.append(mix(x ^ tail))
        return out

    d = chain(d)
    assert [int(x) for x in o.obs_digest] == d
    for _ in range(5):
        o.step()
        d = chain(d)
        assert [int(x) for x in o.obs_digest] == d


@pytest.mark.parametrize("name,N,T,over", [
    ("c2_24x24", 12, 120, dict(max_turns=60, spawn_dmin=4)),
    ("c5b_ffa8", 6, 80, dict(height=12, width=12, spawn_dmin=3, n_cities=4, max_turns=50)),
])
def test_R33_packed_plane_decodes_to_the_three_byte_planes(oracle_mod, name, N, T, over):
    """R33 (NEXT-4): the packed byte is visible << 7 | terrain << 4 | (owner + 2), 0 under fog.  Decoding it here,
    independently, must give back obs_owner / obs_terrain / obs_vis on every cell of sampled play."""
    cfg, _ = workloads.config(name, n_games=N, **over)
    o = oracle_mod.Oracle(cfg)
    o.reset()
    seen_fog = seen_enemy = False
    for t in range(T):
        o.step()
        b = o.field("obs_packed").astype(np.int32)
        vis = b >> 7
        owner = np.where(vis == 1, (b & 15) - 2, -2)
        terrain = np.where(vis == 1, (b >> 4) & 3, 4)
        assert np.array_equal(vis, o.field("obs_vis"))
        assert np.array_equal(owner, o.field("obs_owner"))
        assert np.array_equal(terrain, o.field("obs_terrain"))
        assert ((b & 0x40) == 0).all() and (b[vis == 0] == 0).all()
        seen_fog |= bool((vis == 0).any())
        seen_enemy |= bool(((owner >= 0) & (owner != np.arange(o.P)[None, :, None])).any())
    assert seen_fog and seen_enemy


def test_R34_scoreboard_history_closed_form_and_wrap(oracle_mod):
    """R34 (NEXT-2; "512-step sliding window of the opponent's total army count and ... land count"):
    under all-pass play the general holds 1 + t // 2 + t // 50 at turn t (closed form C1) and land stays 1, so
    slot t mod 512 of the ring must hold exactly that, and after 600 turns slots 0..87 hold turns 512..599."""
    cfg, _ = workloads.config("c1_8x8", n_games=3)
    o = oracle_mod.Oracle(cfg)
    o.reset()
    passes = np.zeros((3, 2), dtype=np.int32)
    for t in range(1, 601):
        o.step(passes)
    h = o.score_hist                                        # [N][512][2P]: (land, army) per player
    for slot in range(512):
        t = slot + 512 if slot + 512 <= 600 else slot
        want_army = 1 + t // 2 + t // 50
        assert (h[:, slot, 0::2] == 1).all() and (h[:, slot, 1::2] == want_army).all(), slot


def test_R34_history_is_the_scoreboard_of_every_turn(oracle_mod):
    """On sampled play with auto-reset: an independent Python log of (turn, land, army_total) after every call must
    equal the ring on the last min(turn + 1, 512) turns of the current episode of every game."""
    cfg, _ = workloads.config("c4_curriculum", n_games=10, height=10, width=10, spawn_dmin=3, spawn_dmax=5,
                              n_cities=3, max_turns=90)
    o = oracle_mod.Oracle(cfg)
    o.reset()
    log = [dict() for _ in range(10)]                       # per game: turn -> (land, army) of the current episode
    ep = o.episode.copy()
    def note():
        for g in range(10):
            if o.episode[g] != ep[g]:
                log[g].clear()
                ep[g] = o.episode[g]
            log[g][int(o.turn[g])] = (o.land[g].copy(), o.army_total[g].copy())
    note()
    for _ in range(300):
        o.step()
        note()
        for g in range(10):
            for t, (land, army) in log[g].items():
                if t > int(o.turn[g]) - 512:
                    assert np.array_equal(o.score_hist[g, t % 512, 0::2], land)
                    assert np.array_equal(o.score_hist[g, t % 512, 1::2], army)
    assert int(o.episodes_done.sum()) > 5 and int(o.wins.sum()) > 0


def test_R39_history_windows_closed_form_wrap_and_enemy_sums(oracle_mod):
    """R39 ("a 512-step sliding window of the opponent's total army count and a matching window of their
    total land count"): under all-pass play every player's army total is 1 + t // 2 + t // 50 at turn t (closed form
    C1) and the land stays 1, so entry i of agent p's windows must read (#enemies) x that closed form at turn
    t - 511 + i, and 0 before turn 0 -- before the ring wraps (t = 300), exactly when it fills (t = 511) and after it
    has wrapped (t = 700); with two players, with three (free-for-all: two enemies) and with 2v2 teams."""
    for P, team, enemies in ((2, 1, 1), (3, 1, 2), (4, 2, 2)):
        cfg, _ = workloads.config("c1_8x8", n_games=2, n_players=P, team_size=team, spawn_dmin=3)
        o = oracle_mod.Oracle(cfg)
        o.reset()
        passes = np.zeros((2, P), dtype=np.int32)
        for t in range(1, 701):
            o.step(passes)
            if t in (300, 511, 700):
                win = o.history_windows()
                assert win.shape == (2, P, 2, 512)
                for i in range(512):
                    tt = t - 511 + i
                    army = enemies * (1 + tt // 2 + tt // 50) if tt >= 0 else 0
                    land = enemies if tt >= 0 else 0
                    assert (win[:, :, 0, i] == army).all() and (win[:, :, 1, i] == land).all(), (P, t, i)


def test_R39_history_windows_follow_an_independent_log(oracle_mod):
    """On sampled play with captures and auto-reset the windows must equal a Python log of the scoreboard kept by the
    test turn by turn (cleared when the episode changes): oldest first, the newest entry is the current scoreboard,
    zeros before the episode's first turn -- per agent, summed over the players off its team (2v2: R38)."""
    cfg, _ = workloads.config("c5a_2v2", n_games=6, height=10, width=10, spawn_dmin=3, n_cities=3, max_turns=60,
                              pass_thr=0)
    o = oracle_mod.Oracle(cfg)
    o.reset()
    P = 4
    log = [dict() for _ in range(6)]
    ep = o.episode.copy()

    def note():
        for g in range(6):
            if o.episode[g] != ep[g]:
                log[g].clear()
                ep[g] = o.episode[g]
            log[g][int(o.turn[g])] = (o.land[g].copy(), o.army_total[g].copy())

    note()
    for step in range(150):
        o.step()
        note()
        if step % 7 == 0 or step > 140:
            win = o.history_windows()
            for g in range(6):
                t = int(o.turn[g])
                for p in range(P):
                    enemy = [q for q in range(P) if q // 2 != p // 2]
                    for i in range(512):
                        tt = t - 511 + i
                        want_a = sum(int(log[g][tt][1][q]) for q in enemy) if tt >= 0 else 0
                        want_l = sum(int(log[g][tt][0][q]) for q in enemy) if tt >= 0 else 0
                        assert win[g, p, 0, i] == want_a and win[g, p, 1, i] == want_l, (step, g, p, i)
    assert int(o.episodes_done.sum()) > 3
