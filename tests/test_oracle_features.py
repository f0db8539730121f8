"""Pins of the oracle's 38-channel feature tensor (NEXT-1; App. A, Table IV; DESIGN R35).
The paper prints no numeric example of the tensor, so the oracle is pinned by what Table IV and arithmetic fix:
identities between channels, a closed form, and an independent history kept by the test from the oracle's OWN plain
observation planes (obs_army / obs_owner / obs_terrain / obs_vis, themselves pinned elsewhere) -- never by re-running
the featuriser's formulas on its own memory."""
import numpy as np
import pytest

import workloads


def play(oracle_mod, cfg, T, actions=None):
    o = oracle_mod.Oracle(cfg)
    o.reset()
    frames = []
    for t in range(T + 1):
        if t > 0:
            o.step(actions)
        f = o.features().copy()
        frames.append(dict(feat=f, turn=o.turn.copy(), episode=o.episode.copy(), land=o.land.copy(),
                           tot=o.army_total.copy(), army=o.field("obs_army").astype(np.int64).copy(),
                           owner=o.field("obs_owner").astype(np.int64).copy(),
                           terrain=o.field("obs_terrain").astype(np.int64).copy(),
                           vis=o.field("obs_vis").astype(np.int64).copy()))
    return o, frames


def test_channel_identities_and_memory_from_an_independent_log(oracle_mod):
    cfg, _ = workloads.config("c4_curriculum", n_games=8, height=9, width=11, spawn_dmin=3, spawn_dmax=5, n_cities=3,
                              max_turns=70)
    o, frames = play(oracle_mod, cfg, 150)
    N, S, HW = 8, o.S, 99
    me = np.arange(2)[None, :, None]
    # the test's own memory, rebuilt from the plain observation planes
    seen = np.zeros((N, 2, S), bool); en_seen = seen.copy(); gens = seen.copy(); cast = seen.copy(); mont = seen.copy()
    last_army = np.zeros((N, 2, S), np.int64); last_turn = np.full((N, 2, S), -1, np.int64)
    own_hist, en_hist = [], []
    resets = 0
    for fr in frames:
        f, vis, owner, army, terrain = fr["feat"], fr["vis"] == 1, fr["owner"], fr["army"], fr["terrain"]
        t = fr["turn"][:, None, None]
        new = (fr["turn"] == 0)
        resets += int(new.sum())
        for arr in (seen, en_seen, gens, cast, mont):
            arr[new] = False
        last_army[new] = 0; last_turn[new] = -1
        own = owner == me
        enemy = vis & (owner == 1 - me)
        neutral = vis & (owner == -1)
        own_a, en_a = np.where(own, army, 0), np.where(enemy, army, 0)
        # Table IV, instantaneous channels
        assert np.array_equal(f[:, :, 0], army) and np.array_equal(f[:, :, 1], own_a) and np.array_equal(f[:, :, 2], en_a)
        assert np.array_equal(f[:, :, 0], f[:, :, 1] + f[:, :, 2] + f[:, :, 3])           # visible army splits by owner
        assert np.array_equal(f[:, :, 9], neutral) and np.array_equal(f[:, :, 10], own)
        assert np.array_equal(f[:, :, 11], enemy) and np.array_equal(f[:, :, 12][:, :, :HW], ~vis[:, :, :HW])
        assert np.array_equal((f[:, :, 9] + f[:, :, 10] + f[:, :, 11] + f[:, :, 12])[:, :, :HW], np.ones((N, 2, HW)))
        # persistent memory
        seen |= vis; en_seen |= enemy; gens |= vis & (terrain == 3); cast |= vis & (terrain == 2); mont |= vis & (terrain == 1)
        for ch, arr in zip(range(4, 9), (seen, en_seen, gens, cast, mont)):
            assert np.array_equal(f[:, :, ch], arr), ch
        assert np.array_equal(f[:, :, 13][:, :, :HW], (~vis & (gens | cast | mont))[:, :, :HW])
        last_army = np.where(enemy, army, last_army); last_turn = np.where(enemy, t, last_turn)
        assert np.array_equal(f[:, :, 20], last_army)
        age = np.where((last_turn < 0) | enemy, 0.0, np.log1p((t - last_turn).astype(np.float64)) / 5.0)
        assert np.abs(f[:, :, 21] - age).max() < 1e-6
        # scalars
        b = f[:, :, :, :HW]                                                                 # broadcast over the board
        assert (b[:, :, 14] == t).all() and np.allclose(b[:, :, 15], (t % 50) / 50.0, atol=1e-7)
        for p in range(2):
            assert (b[:, p, 16] == fr["land"][:, p, None]).all() and (b[:, p, 17] == fr["tot"][:, p, None]).all()
            assert (b[:, p, 18] == fr["land"][:, 1 - p, None]).all() and (b[:, p, 19] == fr["tot"][:, 1 - p, None]).all()
        # delta stacks against the test's own frame log (frames before the episode start count as absent)
        own_hist.append((fr["turn"].copy(), own_a)); en_hist.append((fr["turn"].copy(), en_a))
        for k in range(7):
            for base, hist in ((24, own_hist), (31, en_hist)):
                want = np.zeros((N, 2, S), np.int64)
                if len(hist) >= k + 2:
                    (t1, a1), (t0, a0) = hist[-1 - k], hist[-2 - k]
                    same = (fr["turn"] - k - 1 >= 0) & (t1 == fr["turn"] - k) & (t0 == fr["turn"] - k - 1)
                    want[same] = (a1 - a0)[same]
                assert np.array_equal(f[:, :, base + k], want), (base, k)
        assert (f[:, :, :, HW:] == 0).all()                                                 # stride padding
    assert resets > 12 and en_seen.any() and gens.sum() > 16                                # captures, re-fog, memory


def test_closed_form_under_all_pass_play(oracle_mod):
    """All players pass: the general holds 1 + t // 2 + t // 50 (closed form C1), so own_army_delta[k] at the general
    is the increment of that sequence, the coordinates are col / (W - 1), row / (H - 1), nothing enemy is ever seen."""
    cfg, _ = workloads.config("c1_8x8", n_games=2)
    o = oracle_mod.Oracle(cfg)
    o.reset()
    passes = np.zeros((2, 2), np.int32)
    gen = lambda t: 1 + t // 2 + t // 50 if t >= 0 else 0
    for t in range(0, 120):
        if t > 0:
            o.step(passes)
        f = o.features()
        for g in range(2):
            for p in range(2):
                c = int(o.general_cell[g, p])
                assert f[g, p, 1, c] == gen(t) and f[g, p, 17, c] == gen(t) and f[g, p, 16, c] == 1
                for k in range(7):
                    want = gen(t - k) - gen(t - k - 1) if t - k - 1 >= 0 else 0
                    assert f[g, p, 24 + k, c] == want, (t, k)
                assert f[g, p, 2].sum() == 0 and f[g, p, 5].sum() == 0 and f[g, p, 31:38].sum() == 0
                assert f[g, p, 22, c] == np.float32((c % 8) / 7) and f[g, p, 23, c] == np.float32((c // 8) / 7)
                assert f[g, p, 4].sum() == f[g, p, 0, :64].size - f[g, p, 12, :64].sum()    # seen == visible: nothing moves


@pytest.mark.parametrize("name,P,team_size", [("c5a_2v2", 4, 2), ("c5b_ffa8", 8, 1), ("c5b_ffa8", 3, 1)])
def test_multi_player_features_from_the_plain_observation(oracle_mod, name, P, team_size):
    """R38 (the same observation interface in 1v1, 2v2 and free-for-all): agent = player p, opponent = every
    player off p's team, visibility = the team's.  Pinned against the oracle's plain observation planes (which carry
    the team visibility of P:L83 / R19 and are pinned elsewhere) and the public scoreboard: instantaneous channels,
    the memory rebuilt by the test, the enemy-sum scoreboard entries; the four cell classes now leave out exactly the
    visible cells of allies."""
    cfg, _ = workloads.config(name, n_games=6, height=12, width=13, n_players=P, team_size=team_size, spawn_dmin=3,
                              n_cities=4, max_turns=60)
    o = oracle_mod.Oracle(cfg)
    o.reset()
    N, S, HW = 6, o.S, 12 * 13
    me = np.arange(P)[None, :, None]
    team = np.arange(P) // team_size
    enemy_of = team[:, None] != team[None, :]                          # [agent][other]
    seen = np.zeros((N, P, S), bool); en_seen = seen.copy(); last_army = np.zeros((N, P, S), np.int64)
    last_turn = np.full((N, P, S), -1, np.int64)
    allies_seen = False
    for t in range(140):
        if t:
            o.step()
        f = o.features().copy()
        assert f.shape == (N, P, 38, S)
        new = o.turn == 0
        seen[new] = False; en_seen[new] = False; last_army[new] = 0; last_turn[new] = -1
        vis = o.field("obs_vis").astype(bool)
        owner = o.field("obs_owner").astype(np.int64)
        army = o.field("obs_army").astype(np.int64)
        own = owner == me
        is_player = owner >= 0
        enemy = vis & is_player & enemy_of[np.arange(P)[None, :, None], np.clip(owner, 0, P - 1)]
        ally = vis & is_player & ~own & ~enemy
        allies_seen |= bool(ally.any())
        neutral = vis & (owner == -1)
        assert np.array_equal(f[:, :, 0], army) and np.array_equal(f[:, :, 1], np.where(own, army, 0))
        assert np.array_equal(f[:, :, 2], np.where(enemy, army, 0)) and np.array_equal(f[:, :, 3], np.where(neutral, army, 0))
        assert np.array_equal(f[:, :, 9], neutral) and np.array_equal(f[:, :, 10], own) and np.array_equal(f[:, :, 11], enemy)
        assert np.array_equal(f[:, :, 12][:, :, :HW], ~vis[:, :, :HW])
        assert np.array_equal((f[:, :, 9] + f[:, :, 10] + f[:, :, 11] + f[:, :, 12])[:, :, :HW], 1 - ally[:, :, :HW])
        seen |= vis; en_seen |= enemy
        last_army = np.where(enemy, army, last_army); last_turn = np.where(enemy, o.turn[:, None, None], last_turn)
        assert np.array_equal(f[:, :, 4], seen) and np.array_equal(f[:, :, 5], en_seen)
        assert np.array_equal(f[:, :, 20], last_army)
        age = np.where((last_turn < 0) | enemy, 0.0, np.log1p((o.turn[:, None, None] - last_turn).clip(0)) / 5.0)
        assert np.allclose(f[:, :, 21], age, atol=1e-6)
        land, tot = o.land.astype(np.int64), o.army_total.astype(np.int64)
        for p in range(P):
            assert (f[:, p, 16, :HW] == land[:, p, None]).all() and (f[:, p, 17, :HW] == tot[:, p, None]).all()
            assert (f[:, p, 18, :HW] == land[:, enemy_of[p]].sum(1)[:, None]).all()
            assert (f[:, p, 19, :HW] == tot[:, enemy_of[p]].sum(1)[:, None]).all()
    assert allies_seen == (team_size > 1)
    assert int(o.episodes_done.sum()) > 0


def test_bf16_output_is_the_fp32_tensor_rounded_to_nearest_even(oracle_mod):
    """R37: the bfloat16 variant is the fp32 tensor rounded once, ties to even.  Pinned against torch's own
    float32 -> bfloat16 conversion (a library routine, not the oracle's bit trick) on real play, and on hand-picked
    ties: 257 = 0x4380_8000 is halfway between 256 and 258 -> 256 (even mantissa); 259 -> 260; 32767 -> 32768."""
    import torch
    cfg, _ = workloads.config("c4_curriculum", n_games=6, height=9, width=11, spawn_dmin=3, spawn_dmax=5, n_cities=3,
                              max_turns=70)
    o = oracle_mod.Oracle(cfg)
    o.reset()
    for t in range(120):
        if t:
            o.step()
        if t % 10 == 0:                     # make large armies appear: bf16 cannot hold them exactly
            big = np.minimum(o.army[:, :99].astype(np.int32) * 7 + 250, 30000).astype(np.int16)
            o.army[:, :99] = np.where(o.owner[:, :99] >= 0, big, o.army[:, :99])
            o.observe()
        f16 = o.features(bf16=True).copy()
        f32 = o.feat.copy()
        want = torch.from_numpy(f32).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
        assert np.array_equal(f16, want)
    assert (f32 > 256).any()
    for val, bits in ((257.0, 0x4380), (259.0, 0x4382), (32767.0, 0x4700), (1.0, 0x3F80), (0.0, 0)):
        got = torch.tensor([val], dtype=torch.float32).to(torch.bfloat16).view(torch.int16).item() & 0xFFFF
        assert got == bits


def test_hand_worked_example_W12(oracle_mod):
    """tests/golden/features_worked_example.txt: four turns on a 2 x 3 board, every channel of three (turn, player)
    views written out by hand from Table IV (values, memory, fog, age, scoreboard, coordinates, both delta stacks)."""
    import os
    from helpers import hand_board, act, DOWN, LEFT, UP
    PL, MT, CT, GN = 0, 1, 2, 3
    o = hand_board(oracle_mod, 2, 3, 2, {(0, 0): (GN, 0, 5), (0, 1): (PL, 0, 3), (0, 2): (MT, -1, 0),
                                         (1, 0): (CT, -1, 42), (1, 2): (GN, 1, 7)}, turn=0)
    moves = [None, (act(0, 1, 3, DOWN), 0), (0, act(1, 2, 3, LEFT)), (0, act(1, 1, 3, UP))]
    frames = []
    for mv in moves:
        if mv is not None:
            o.step(np.array([mv], dtype=np.int32))
        frames.append(o.features().copy())
    assert int(o.turn[0]) == 3
    want = {}
    path = os.path.join(os.path.dirname(__file__), "golden", "features_worked_example.txt")
    for line in open(path):
        if line.startswith("#") or not line.strip():
            continue
        tok = line.split()
        want.setdefault((int(tok[0]), int(tok[1])), {})[int(tok[2])] = np.array([float(x) for x in tok[3:]], np.float32)
    assert sorted(want) == [(0, 1), (1, 1), (3, 0)]
    for (fr, p), chans in want.items():
        for ch in range(38):
            got = frames[fr][0, p, ch, :6]
            exp = chans.get(ch, np.zeros(6, np.float32))
            if ch == 21:
                assert np.allclose(got, exp, atol=1e-6), (fr, p, ch, got)
            else:
                assert np.array_equal(got, exp), (fr, p, ch, got, exp)
        assert not frames[fr][0, p, :, 6:].any()                 # stride padding is zero


def test_padded_border_is_a_known_mountain(oracle_mod):
    """Table IV ch 8 "visible mountains U known padded border" and ch 13 "... or unseen padded border" on official
    maps with a playable area smaller than the board (R36): from turn 0 on, every cell outside the playable
    rectangle is in the mountain memory whether or not it has been seen; in fog it counts as a known structure.  The
    border is re-derived here from the terrain plane (all-mountain suffix rows / columns agree with play_size), the
    rest of ch 8 / ch 13 from the plain observation planes."""
    cfg, _ = workloads.config("official_23x23", n_games=12, max_turns=40, spawn_dmin=6)
    o = oracle_mod.Oracle(cfg)
    o.reset()
    H = W = 23
    HW = H * W
    seen_mtn = np.zeros((12, 2, HW), bool)
    seen_str = np.zeros((12, 2, HW), bool)
    saw_small = False
    for t in range(90):
        if t:
            o.step()
        f = o.features().copy()
        new = o.turn == 0
        seen_mtn[new] = False
        seen_str[new] = False
        ph, pw = o.play_size[:, 0].astype(int), o.play_size[:, 1].astype(int)
        rr, cc = np.divmod(np.arange(HW), W)
        border = (rr[None, :] >= ph[:, None]) | (cc[None, :] >= pw[:, None])           # [N][HW]
        terr = o.terrain[:, :HW]
        assert (terr[border] == 1).all()                                                # the padding is mountains
        assert ((ph >= 18) & (ph <= 23) & (pw >= 18) & (pw <= 23)).all()
        saw_small |= bool(border.any())
        vis = o.field("obs_vis")[:, :, :HW] == 1
        ot = o.field("obs_terrain")[:, :, :HW]
        seen_mtn |= vis & (ot == 1)
        seen_str |= vis & ((ot == 2) | (ot == 3))
        want8 = seen_mtn | border[:, None, :]
        assert np.array_equal(f[:, :, 8, :HW] == 1, want8)
        want13 = ~vis & (want8 | seen_str)
        assert np.array_equal(f[:, :, 13, :HW] == 1, want13)
        # a border cell that has never been seen is already known at turn 0
        if t == 0:
            unseen_border = border[:, None, :] & ~vis
            assert unseen_border.any() and (f[:, :, 13, :HW][unseen_border] == 1).all()
    assert saw_small and int(o.episodes_done.sum()) > 0
    # full boards: no border, ch 8 is the seen mountains only (the synthetic generator reports H x W)
    cfg2, _ = workloads.config("c2_24x24", n_games=3)
    o2 = oracle_mod.Oracle(cfg2)
    o2.reset()
    assert (o2.play_size == 24).all()
    f2 = o2.features()
    vis2 = o2.field("obs_vis")[:, :, :576] == 1
    assert np.array_equal(f2[:, :, 8, :576] == 1, vis2 & (o2.field("obs_terrain")[:, :, :576] == 1))
