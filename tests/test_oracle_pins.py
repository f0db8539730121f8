"""Pins for the CPU oracle that do not come from the oracle itself.

Known-answer vectors of published generators (tests/golden/), and hand-worked examples W1..W11
derived by hand from PAPER.md section IV under the readings R1..R32 of DESIGN.md.
Every expected number below was worked out on paper from the cited rule, not by running code.
"""
import os

import numpy as np
import pytest

from helpers import DOWN, LEFT, PASS, RIGHT, UP, act, cell, hand_board

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
PL, MT, CT, GN = 0, 1, 2, 3


def _rows(name):
    with open(os.path.join(GOLDEN, name)) as f:
        return [l.split() for l in f if l.strip() and not l.startswith("#")]


def test_philox_known_answers(oracle_mod):
    """P1: Random123 KAT rows for philox4x32-10."""
    rows = _rows("philox_kat.txt")
    assert len(rows) == 3
    for row in rows:
        v = [int(x, 16) for x in row]
        assert oracle_mod.philox4x32_10(v[0:4], v[4:6]) == tuple(v[6:10])


def test_splitmix64_known_answers(oracle_mod):
    """mix64 is the splitmix64 finaliser: output n of seed 0 is mix64(n * golden gamma)."""
    outs = [int(r[0], 16) for r in _rows("splitmix64_seed0.txt")]
    for n, want in enumerate(outs, start=1):
        assert oracle_mod.mix64((n * 0x9E3779B97F4A7C15) & (2**64 - 1)) == want
        assert oracle_mod.digest_key(n - 1) == want | 1


def _two_generals(extra, H=3, W=3, turn=0, **cfg):
    cells = {(0, 0): (GN, 0, 1), (H - 1, W - 1): (GN, 1, 1)}
    cells.update(extra)
    return cells, dict(H=H, W=W, turn=turn, **cfg)


def _board(oracle_mod, extra, H=3, W=3, turn=0, P=2, **cfg):
    cells, _ = _two_generals(extra, H, W)
    return hand_board(oracle_mod, H, W, P, cells, turn=turn, **cfg)


def test_W1_all_but_one_onto_empty(oracle_mod):
    o = _board(oracle_mod, {(1, 0): (PL, 0, 5)})
    o.step([[act(1, 0, 3, RIGHT), PASS]])
    assert cell(o, 1, 0) == (PL, 0, 1)
    assert cell(o, 1, 1) == (PL, 0, 4)
    assert int(o.turn[0]) == 1 and int(o.done[0, 0]) == 0


@pytest.mark.parametrize("army,sent,kept", [(7, 3, 4), (2, 1, 1), (3, 1, 2), (100, 50, 50)])
def test_W2_half_split_rounds_down(oracle_mod, army, sent, kept):
    """R4: 'exactly half' of an odd stack sends floor(a/2)."""
    o = _board(oracle_mod, {(1, 0): (PL, 0, army)})
    o.step([[act(1, 0, 3, RIGHT, half=1), PASS]])
    assert cell(o, 1, 0) == (PL, 0, kept)
    assert cell(o, 1, 1) == (PL, 0, sent)


@pytest.mark.parametrize("half", [0, 1])
def test_W2_army_one_cannot_move(oracle_mod, half):
    """R5: 'all-but-one' needs at least 2 units."""
    o = _board(oracle_mod, {(1, 0): (PL, 0, 1)})
    before = (o.army.copy(), o.owner.copy())
    o.step([[act(1, 0, 3, RIGHT, half), PASS]])
    assert np.array_equal(o.army, before[0]) and np.array_equal(o.owner, before[1])


def test_W3_merge_onto_own_cell(oracle_mod):
    o = _board(oracle_mod, {(1, 0): (PL, 0, 5), (1, 1): (PL, 0, 3)})
    o.step([[act(1, 0, 3, RIGHT), PASS]])
    assert cell(o, 1, 0) == (PL, 0, 1) and cell(o, 1, 1) == (PL, 0, 7)


@pytest.mark.parametrize("defender,want_owner,want_army", [(3, 0, 1), (4, 1, 0), (7, 1, 3)])
def test_W4_combat_by_subtraction(oracle_mod, defender, want_owner, want_army):
    """stacks cancel one-for-one, larger survives with the difference, ties keep the owner."""
    o = _board(oracle_mod, {(1, 0): (PL, 0, 5), (1, 1): (PL, 1, defender)})
    o.step([[act(1, 0, 3, RIGHT), PASS]])
    assert cell(o, 1, 0) == (PL, 0, 1)
    assert cell(o, 1, 1) == (PL, want_owner, want_army)
    assert int(o.done[0, 0]) == 0


@pytest.mark.parametrize("defender,captured,want_army", [(3, True, 1), (4, False, 0), (7, False, 3)])
def test_W4_general_needs_strictly_more(oracle_mod, defender, captured, want_army):
    """R12: a tie does not capture a general."""
    cells = {(0, 0): (GN, 0, 1), (1, 0): (PL, 0, 5), (1, 1): (GN, 1, defender)}
    o = hand_board(oracle_mod, 3, 3, 2, cells, turn=0)
    o.step([[act(1, 0, 3, RIGHT), PASS]])
    if captured:
        assert cell(o, 1, 1) == (CT, 0, want_army)          # general becomes a castle
        assert int(o.done[0, 0]) == 1 and int(o.winner[0, 0]) == 0
        assert o.reward[0, 0].tolist() == [1, -1]
        assert int(o.alive[0]) == 0b01 and int(o.general_cell[0, 1]) == -1
    else:
        assert cell(o, 1, 1) == (GN, 1, want_army)
        assert int(o.done[0, 0]) == 0 and o.reward[0, 0].tolist() == [0, 0]


@pytest.mark.parametrize("stack,want", [(51, (CT, 0, 5)), (46, (CT, -1, 0)), (47, (CT, 0, 1))])
def test_W5_neutral_castle_is_paid_down(oracle_mod, stack, want):
    """P:L87 + R9: a neutral castle fights like an enemy cell; a tie leaves it neutral with 0."""
    o = _board(oracle_mod, {(1, 0): (PL, 0, stack), (1, 1): (CT, -1, 45)})
    o.step([[act(1, 0, 3, RIGHT), PASS]])
    assert cell(o, 1, 1) == want
    # turn is now 1; the next step makes it 2 (even): an owned castle produces, a neutral one does not
    o.step([[PASS, PASS]])
    t, ow, a = want
    assert cell(o, 1, 1) == (t, ow, a + (1 if ow == 0 else 0))


def test_W6_contested_cell_lower_index_first(oracle_mod):
    """R6: sequential resolution in ascending player index."""
    o = _board(oracle_mod, {(1, 0): (PL, 0, 4), (1, 2): (PL, 1, 6)})
    o.step([[act(1, 0, 3, RIGHT), act(1, 2, 3, LEFT)]])
    assert cell(o, 1, 0) == (PL, 0, 1)
    assert cell(o, 1, 1) == (PL, 1, 2)
    assert cell(o, 1, 2) == (PL, 1, 1)


def test_W6_rotate_priority_flag(oracle_mod):
    """rule_flags bit ROTATE_PRIORITY: the first mover is turn % P (turn before the increment)."""
    o = _board(oracle_mod, {(1, 0): (PL, 0, 4), (1, 2): (PL, 1, 6)}, turn=1,
               rule_flags=oracle_mod.RULE_ROTATE_PRIORITY)
    o.step([[act(1, 0, 3, RIGHT), act(1, 2, 3, LEFT)]])
    # P1 first: 5 onto empty -> P1 5; then P0's 3 against 5 -> P1 2.  Same cell result, but turn 2 is
    # even so generals grow; check the contested cell and sources
    assert cell(o, 1, 1) == (PL, 1, 2)
    o2 = _board(oracle_mod, {(1, 0): (PL, 0, 5), (1, 1): (PL, 1, 5)}, turn=1,
                rule_flags=oracle_mod.RULE_ROTATE_PRIORITY)
    o2.step([[act(1, 0, 3, RIGHT), act(1, 1, 3, LEFT)]])
    # P1 first: 4 against P0's 5 -> P0 keeps (1,0) with 1; P0's move is now void (army 1)
    assert cell(o2, 1, 0) == (PL, 0, 1) and cell(o2, 1, 1) == (PL, 1, 1)


def test_W7_swap_revalidates_second_mover(oracle_mod):
    """R7: a later mover is re-validated on the board as it is when applied."""
    o = _board(oracle_mod, {(1, 0): (PL, 0, 5), (1, 1): (PL, 1, 5)})
    o.step([[act(1, 0, 3, RIGHT), act(1, 1, 3, LEFT)]])
    assert cell(o, 1, 0) == (PL, 0, 1)
    assert cell(o, 1, 1) == (PL, 1, 1)


W8_CELLS = {(0, 0): (GN, 0, 3), (3, 2): (PL, 0, 10), (3, 3): (GN, 1, 4), (2, 3): (PL, 1, 7),
            (1, 3): (PL, 1, 1), (2, 2): (PL, 1, 2), (0, 3): (CT, -1, 45), (1, 1): (MT, -1, 0)}


@pytest.mark.parametrize("floor", [False, True])
def test_W8_general_capture_transfers_land_and_half_army(oracle_mod, floor):
    """P:L97 + R11: all cells to the captor with half the army (per cell, rounded up; FLOOR flag
    rounds down), general -> castle, loser's own move the same turn is void (R7)."""
    flags = oracle_mod.RULE_CAPTURE_HALF_FLOOR if floor else 0
    o = hand_board(oracle_mod, 4, 4, 2, W8_CELLS, turn=10, rule_flags=flags)
    o.step([[act(3, 2, 4, RIGHT), act(2, 3, 4, LEFT)]])
    assert int(o.turn[0]) == 11
    assert cell(o, 3, 2) == (PL, 0, 1)
    assert cell(o, 3, 3) == (CT, 0, 5)
    assert cell(o, 2, 3) == (PL, 0, 3 if floor else 4)
    assert cell(o, 1, 3) == (PL, 0, 0 if floor else 1)
    assert cell(o, 2, 2) == (PL, 0, 1)
    assert cell(o, 0, 3) == (CT, -1, 45) and cell(o, 1, 1) == (MT, -1, 0)
    assert o.land[0].tolist() == [6, 0]
    assert o.army_total[0].tolist() == [13 if floor else 15, 0]
    assert o.reward[0, 0].tolist() == [1, -1]
    assert int(o.done[0, 0]) == 1 and int(o.winner[0, 0]) == 0
    assert int(o.alive[0]) == 1 and o.general_cell[0].tolist() == [0, -1]
    assert int(o.episodes_done[0]) == 1 and o.wins[0].tolist() == [1, 0]
    # the winner now sees everything near its 6 cells; the loser owns nothing and sees nothing
    assert int(o.obs_vis[0, 0, 1].sum()) == 0
    assert (o.obs_owner[0, 0, 1, :16] == -2).all() and (o.obs_terrain[0, 0, 1, :16] == 4).all()


def test_W9_moves_then_growth_then_observation(oracle_mod):
    """R1/R3/R32: turn 1 -> 2 is even, growth comes after the move, the observation shows the result."""
    cells = {(0, 0): (GN, 0, 2), (2, 2): (GN, 1, 1)}
    o = hand_board(oracle_mod, 3, 3, 2, cells, turn=1)
    o.step([[act(0, 0, 3, RIGHT), PASS]])
    assert int(o.turn[0]) == 2
    assert cell(o, 0, 0) == (GN, 0, 2)            # 2 - 1 sent + 1 grown
    assert cell(o, 0, 1) == (PL, 0, 1)            # plain cells do not grow on even turns
    assert cell(o, 2, 2) == (GN, 1, 2)
    vis0 = o.obs_vis[0, 0, 0, :9].reshape(3, 3)
    vis1 = o.obs_vis[0, 0, 1, :9].reshape(3, 3)
    assert vis0.tolist() == [[1, 1, 1], [1, 1, 1], [0, 0, 0]]
    assert vis1.tolist() == [[0, 0, 0], [0, 1, 1], [0, 1, 1]]
    assert o.obs_army[0, 0, 0, :9].tolist() == [2, 1, 0, 0, 0, 0, 0, 0, 0]
    assert o.obs_owner[0, 0, 0, :9].tolist() == [0, 0, -1, -1, -1, -1, -2, -2, -2]
    assert o.obs_terrain[0, 0, 0, :9].tolist() == [3, 0, 0, 0, 0, 0, 4, 4, 4]
    assert o.obs_army[0, 0, 1, :9].tolist() == [0, 0, 0, 0, 0, 0, 0, 0, 2]
    assert o.land[0].tolist() == [2, 1] and o.army_total[0].tolist() == [3, 2]


def _team_board(oracle_mod, target):
    # 5x5, 2v2: teams {0,1} and {2,3}; generals in the corners
    cells = {(0, 0): (GN, 0, 1), (0, 4): (GN, 2, 1), (4, 0): (GN, 3, 1), (2, 0): (PL, 0, 6)}
    cells[(2, 1)] = target
    if target[0] != GN:
        cells[(4, 4)] = (GN, 1, 1)
    return hand_board(oracle_mod, 5, 5, 4, cells, turn=0, team_size=2)


def test_W10_team_move_onto_ally(oracle_mod):
    """moving onto an ally's cell takes ownership and pools the units."""
    o = _team_board(oracle_mod, (PL, 1, 3))
    o.step([[act(2, 0, 5, RIGHT), PASS, PASS, PASS]])
    assert cell(o, 2, 0) == (PL, 0, 1) and cell(o, 2, 1) == (PL, 0, 8)
    assert int(o.done[0, 0]) == 0


def test_W10_ally_general_keeps_its_owner(oracle_mod):
    """R19: units pool onto an ally's general but the general does not change hands."""
    o = _team_board(oracle_mod, (GN, 1, 3))
    o.step([[act(2, 0, 5, RIGHT), PASS, PASS, PASS]])
    assert cell(o, 2, 0) == (PL, 0, 1) and cell(o, 2, 1) == (GN, 1, 8)
    assert int(o.alive[0]) == 0b1111 and int(o.done[0, 0]) == 0


def test_W10_shared_team_vision(oracle_mod):
    o = _team_board(oracle_mod, (PL, 1, 3))
    assert np.array_equal(o.obs_vis[0, 0, 0], o.obs_vis[0, 0, 1])
    assert np.array_equal(o.obs_vis[0, 0, 2], o.obs_vis[0, 0, 3])
    assert not np.array_equal(o.obs_vis[0, 0, 0], o.obs_vis[0, 0, 2])


def test_W11_int16_saturation(oracle_mod):
    """R21: additions clamp at 32767 and are counted."""
    o = _board(oracle_mod, {(1, 0): (PL, 0, 21), (1, 1): (PL, 0, 32760)})
    o.step([[act(1, 0, 3, RIGHT), PASS]])
    assert cell(o, 1, 1) == (PL, 0, 32767) and int(o.sat_events[0]) == 1
    assert cell(o, 1, 0) == (PL, 0, 1)


def test_team_elimination_and_last_team_standing(oracle_mod):
    """the team loses when both generals are captured; everyone on the winning team gets +1,
    including an eliminated member (R20)."""
    cells = {(0, 0): (GN, 0, 1), (0, 2): (GN, 2, 1), (0, 1): (PL, 0, 9),     # P0 next to P2's general
             (2, 2): (GN, 3, 1), (2, 1): (PL, 1, 9), (2, 0): (GN, 1, 1),
             (1, 2): (PL, 3, 4)}
    o = hand_board(oracle_mod, 3, 3, 4, cells, turn=0, team_size=2)
    o.step([[act(0, 1, 3, RIGHT), PASS, PASS, PASS]])          # P0 captures P2
    assert int(o.alive[0]) == 0b1011 and int(o.done[0, 0]) == 0
    assert cell(o, 0, 2) == (CT, 0, 7)
    o.step([[PASS, act(2, 1, 3, RIGHT), PASS, PASS]])          # P1 captures P3 (turn 2: P3 grew? no,
    # growth happens after moves: P3's general still has 1 when P1's 8 arrive)
    assert int(o.alive[0]) == 0b0011
    assert int(o.done[0, 0]) == 1 and int(o.winner[0, 0]) == 0
    assert o.reward[0, 0].tolist() == [1, 1, -1, -1]
    # P3's other cell (1,2)=4 went to the captor P1 with ceil(4/2)=2
    assert cell(o, 1, 2) == (PL, 1, 2)


def test_ffa_capture_keeps_playing(oracle_mod):
    """P:L97 FFA: capture transfers cells, game continues until the last general stands."""
    cells = {(0, 0): (GN, 0, 1), (0, 1): (PL, 0, 5), (0, 2): (GN, 1, 2), (2, 2): (GN, 2, 1),
             (1, 2): (PL, 1, 9)}
    o = hand_board(oracle_mod, 3, 3, 3, cells, turn=0)
    o.step([[act(0, 1, 3, RIGHT), PASS, PASS]])
    assert int(o.done[0, 0]) == 0 and int(o.alive[0]) == 0b101
    assert cell(o, 0, 2) == (CT, 0, 2) and cell(o, 1, 2) == (PL, 0, 5)
    assert o.reward[0, 0].tolist() == [0, 0, 0]
    assert o.land[0].tolist() == [4, 0, 1]


def test_truncation_and_frozen_game(oracle_mod):
    """R16/R31: max_turns truncates with zero rewards; without auto-reset the game freezes."""
    o = _board(oracle_mod, {}, turn=8, max_turns=10, auto_reset=0)
    o.step([[PASS, PASS]])
    assert int(o.done[0, 0]) == 0
    o.step([[PASS, PASS]])
    assert int(o.turn[0]) == 10 and int(o.done[0, 0]) == 2 and int(o.winner[0, 0]) == -1
    assert o.reward[0, 0].tolist() == [0, 0] and int(o.truncations[0]) == 1
    army = o.army.copy()
    o.step([[act(0, 0, 3, RIGHT), PASS]])
    assert int(o.turn[0]) == 10 and int(o.done[0, 0]) == 2 and np.array_equal(o.army, army)
    assert int(o.episodes_done[0]) == 1


def test_invalid_and_out_of_range_actions_are_passes(oracle_mod):
    o = _board(oracle_mod, {(1, 1): (PL, 0, 5), (0, 1): (MT, -1, 0)})
    before = o.army.copy()
    for a in (-1, 9 * 9, 2**31 - 1, act(1, 1, 3, UP),        # into the mountain
              act(0, 0, 3, UP), act(0, 0, 3, LEFT),          # off the board
              act(2, 2, 3, LEFT),                            # not P0's cell
              act(1, 2, 3, LEFT)):                           # neutral cell
        o.step([[a, PASS]])
        exp = before.copy()
        assert np.array_equal(o.army[0, :9] - exp[0, :9] >= 0, np.ones(9, bool))
        assert np.array_equal(o.owner[0, :9] == 0, [1, 0, 0, 0, 1, 0, 0, 0, 0])
    # a legal move next to them still works
    o.step([[act(1, 1, 3, DOWN), PASS]])
    assert cell(o, 2, 1)[1] == 0


def test_W13_unclaimed_or_second_general_is_a_castle(oracle_mod):
    """R40: the rules never produce a GENERAL cell that is not the recorded general of its owner; a
    hand-written state that holds one -- an owner-less general ("unclaimed castles/generals", Table IV ch. 3, is the
    paper's only word on it, with no rule attached), or a second GENERAL cell of a player -- is normalised by the
    observe entry point: the cell becomes a CITY.  Taking it is then castle arithmetic by hand: 5 - 1 = 4 sent onto
    2 defenders leaves 2 and the cell changes hands; nobody is eliminated, no land moves, the game goes on; taking
    the second 'general' of player 1 (a castle now) eliminates nobody either."""
    cells = {(0, 0): (GN, 0, 5), (2, 2): (GN, 1, 3), (0, 1): (GN, -1, 2), (2, 0): (GN, 1, 1), (1, 0): (PL, 0, 6)}
    o = hand_board(oracle_mod, 3, 3, 2, cells, turn=0)
    assert cell(o, 0, 1) == (CT, -1, 2) and cell(o, 2, 0) == (CT, 1, 1)          # normalised
    assert cell(o, 0, 0)[0] == GN and cell(o, 2, 2)[0] == GN
    assert o.general_cell[0].tolist() == [0, 8] and int(o.alive[0]) == 0b11
    o.step([[act(0, 0, 3, RIGHT), PASS]])
    assert cell(o, 0, 1) == (CT, 0, 2) and cell(o, 0, 0) == (GN, 0, 1)
    assert int(o.alive[0]) == 0b11 and int(o.done[0, 0]) == 0 and o.land[0].tolist() == [3, 2]
    o.step([[act(1, 0, 3, DOWN), PASS]])                                         # 5 onto player 1's castle of 1
    assert cell(o, 2, 0) == (CT, 0, 5) and int(o.alive[0]) == 0b11 and int(o.done[0, 0]) == 0   # 4 left, +1 (turn 2)
    assert cell(o, 2, 2) == (GN, 1, 4) and o.land[0].tolist() == [4, 1]


def test_invalid_actions_counter_by_hand(oracle_mod):
    """"Invalid game actions are not errors -- they are passes; a device counter invalid_actions is
    diagnostic only."  Every kind of rejected non-pass action counts once, passes and applied moves never: worked out
    by hand on a 3x3 board (player 0: general (0,0) with 5 and a plain cell (1,0) with 1; player 1: general (2,2)
    with 3 and (1,2) with 4; a mountain at (0,1))."""
    MT = oracle_mod.T_MOUNTAIN
    cells = {(0, 0): (GN, 0, 5), (1, 0): (PL, 0, 1), (2, 2): (GN, 1, 3), (1, 2): (PL, 1, 4), (0, 1): (MT, -1, 0)}
    steps = [
        ([PASS, PASS], 0),                                            # cell 0, k 0
        ([4 * 9, 7 * 9], 0),                                          # k = 0 on other cells: still a pass (R22)
        ([-1, 9 * 9], 2),                                             # both out of range
        ([act(0, 0, 3, RIGHT), act(1, 2, 3, RIGHT)], 2),              # into the mountain; off the board
        ([act(1, 0, 3, RIGHT), act(0, 0, 3, DOWN)], 2),               # army 1 < 2; not player 1's cell
        ([act(0, 0, 3, UP), act(1, 1, 3, LEFT)], 2),                  # off the board; a neutral cell
        ([act(0, 0, 3, DOWN), act(1, 2, 3, LEFT)], 0),                # both applied
        ([PASS, act(1, 2, 3, LEFT)], 1),                              # (1,2) was emptied to 1 by the move before
    ]
    o = hand_board(oracle_mod, 3, 3, 2, cells, turn=1)
    total = 0
    for actions, bad in steps:
        o.step([actions])
        total += bad
        assert int(o.invalid_actions[0]) == total, (actions, int(o.invalid_actions[0]), total)
    # an action made invalid by an EARLIER mover of the same turn (R7): player 0 takes (1,1) first with 4 > 3,
    # player 1's move out of (1,1) is then not from its own cell any more
    o = hand_board(oracle_mod, 3, 3, 2, {(0, 0): (GN, 0, 1), (2, 2): (GN, 1, 1), (1, 0): (PL, 0, 5), (1, 1): (PL, 1, 3)}, turn=1)
    o.step([[act(1, 0, 3, RIGHT), act(1, 1, 3, UP)]])
    assert cell(o, 1, 1) == (PL, 0, 1) and int(o.invalid_actions[0]) == 1
    o.reset()
    assert int(o.invalid_actions[0]) == 0
