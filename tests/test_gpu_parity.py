"""Parity of the CUDA path (through the C ABI) with the CPU oracle: bit-exact on every state plane,
observation plane, scoreboard, reward, done flag, accumulator and digest, on the same seeded inputs.
All of this is integer work, so the bar is equality (BASELINE.json north_star)."""
import numpy as np
import pytest

from helpers import DOWN, LEFT, OUT_FIELDS, PASS, RIGHT, STATE_FIELDS, UP, act
import workloads

pytestmark = pytest.mark.gpu

PL, MT, CT, GN = 0, 1, 2, 3
ALL_FIELDS = STATE_FIELDS + OUT_FIELDS


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device")
    import paper_2606_23348_b200 as g
    g.load_library()
    return g


def compare(env, o, fields=ALL_FIELDS, digest=True, slot=0, oslot=0, where=""):
    env.torch.cuda.synchronize()
    for f in fields:
        got = env.field(f, slot)
        want = np.asarray(getattr(o, f))
        if f in OUT_FIELDS or f == "obs_packed":
            want = want[oslot]
        if not np.array_equal(got, want.reshape(got.shape)):
            bad = np.argwhere(got != want.reshape(got.shape))
            raise AssertionError(f"{where}: field {f} differs at {bad[:5].tolist()} "
                                 f"got {got[tuple(bad[0])]} want {want.reshape(got.shape)[tuple(bad[0])]}")
    if digest:
        assert np.array_equal(env.field("obs_digest"), o.obs_digest), f"{where}: digest"


def make_pair(gpu, oracle_mod, cfg, k_slots=1):
    env = gpu.GeneralsEnv(cfg, k_slots=k_slots)
    o = oracle_mod.Oracle(cfg, every_step_K=k_slots if k_slots > 1 else 0)
    return env, o


# ------------------------------------------------------------------------------- config 1 in full
def test_config1_sampler_every_step(gpu, oracle_mod):
    """BASELINE config 1: 1v1 8x8, 64 games, 300 steps, built-in sampler; every tensor every step."""
    cfg, T = workloads.config("c1_8x8")
    env, o = make_pair(gpu, oracle_mod, cfg)
    env.reset()
    o.reset()
    compare(env, o, where="reset")
    for t in range(T):
        env.step()
        acts = o.step(want_actions=True)
        compare(env, o, where=f"step {t}")
        assert np.array_equal(env.field("actions_out"), acts)
    assert env.global_step == T
    assert int(o.done[0].astype(bool).sum()) > 0          # some games end inside 300 steps


def test_config1_explicit_actions(gpu, oracle_mod):
    """Explicit action path with uniformly random (mostly invalid) and garbage actions."""
    import torch
    cfg, T = workloads.config("c1_8x8")
    env, o = make_pair(gpu, oracle_mod, cfg)
    env.reset()
    o.reset()
    rng = np.random.default_rng(5)
    for t in range(120):
        if t % 3 == 0:
            a = workloads.random_actions(rng, 64, 2, 8, 8)
        else:                                              # valid moves, so that the boards evolve
            a = o.sample()
            o.global_step += 1
            flip = rng.random(a.shape) < 0.1
            a = np.where(flip, workloads.random_actions(rng, 64, 2, 8, 8), a).astype(np.int32)
        env.step(torch.from_numpy(a).to(env.device))
        o.step(a)
        compare(env, o, where=f"step {t}")


# ------------------------------------------------------------------------------- configs 2..5, shrunk N
@pytest.mark.parametrize("name,N,T,over", [
    ("c2_24x24", 96, 260, dict(max_turns=120)),
    ("c4_curriculum", 80, 400, dict(max_turns=300)),
    ("c5a_2v2", 40, 260, dict(max_turns=200)),
    ("c5b_ffa8", 40, 260, dict(max_turns=200)),
    ("c5b_ffa8", 24, 200, dict(n_players=3, height=12, width=13, spawn_dmin=5, n_cities=4, max_turns=150)),
    ("c2_24x24", 33, 200, dict(height=5, width=7, spawn_dmin=3, n_cities=2, max_turns=90)),
    ("c2_24x24", 20, 150, dict(height=32, width=32, rule_flags=7, max_turns=100)),
    ("c1_8x8", 20, 150, dict(height=1, width=32, spawn_dmin=8, n_cities=2)),
    ("c1_8x8", 20, 150, dict(height=31, width=3, spawn_dmin=8, n_cities=2, auto_reset=1, max_turns=70)),
])
def test_sampled_play_matches_oracle(gpu, oracle_mod, name, N, T, over):
    """Configs 2-5 at reduced N (several CTAs plus a ragged tail), every tensor compared every step."""
    cfg, _ = workloads.config(name, n_games=N, **over)
    env, o = make_pair(gpu, oracle_mod, cfg)
    env.reset()
    o.reset()
    compare(env, o, where="reset")
    for t in range(T):
        env.step()
        o.step()
        compare(env, o, where=f"{name} step {t}")
    if cfg["max_turns"]:
        assert int(o.episodes_done.sum()) > 0


def test_captures_happen_and_match(gpu, oracle_mod):
    """Config 4's biased policy at short spawn distances drives general captures + land transfer."""
    cfg, _ = workloads.config("c4_curriculum", n_games=128, spawn_dmin=3, spawn_dmax=5, height=10, width=10,
                              n_cities=3, max_turns=400)
    env, o = make_pair(gpu, oracle_mod, cfg)
    env.reset()
    o.reset()
    for t in range(500):
        env.step()
        o.step()
        if t % 10 == 0:
            compare(env, o, where=f"step {t}")
    compare(env, o, where="end")
    assert int(o.wins.sum()) > 20                          # real captures, not truncations


# ------------------------------------------------------------------------------- board-specialised kernels
@pytest.mark.parametrize("name,N,T,over", [
    ("c2_24x24", 101, 230, dict(max_turns=110)),
    ("c4_curriculum", 75, 300, dict(max_turns=200)),
    ("c1_8x8", 77, 200, dict(auto_reset=1, max_turns=80)),
    ("c5a_2v2", 37, 230, dict(max_turns=150)),
    ("c5b_ffa8", 37, 230, dict(max_turns=150)),
])
def test_specialised_step_kernels_match_oracle(gpu, oracle_mod, name, N, T, over):
    """gen_step as bench.py times it (bitboard cache, no digest buffer): the register-resident kernel compiled
    for the paper-sized board against the oracle, every tensor every step; the same kernel's generic
    instantiation and the staged kernel must agree too."""
    cfg, _ = workloads.config(name, n_games=N, **over)
    env = gpu.GeneralsEnv(cfg, digest=False)
    env.set_generic(False, -1)                              # also for 8 players, where the default is the staged kernel
    gen = gpu.GeneralsEnv(cfg, digest=False)
    gen.set_generic(True, -1)
    stg = gpu.GeneralsEnv(cfg, digest=False, bitboards=False)
    o = oracle_mod.Oracle(cfg)
    for e in (env, gen, stg):
        e.reset()
    o.reset()
    for t in range(T):
        for e in (env, gen, stg):
            e.step()
        o.step()
        compare(env, o, digest=False, where=f"{name} specialised step {t}")
        if t % 16 == 0:
            compare(gen, o, digest=False, where=f"{name} generic step {t}")
            compare(stg, o, digest=False, where=f"{name} staged step {t}")
    assert env.last_launch_specialised and env.last_launch_register_resident      # also under the biased policy (R25)
    assert not gen.last_launch_specialised and gen.last_launch_register_resident
    assert not stg.last_launch_register_resident
    assert int(o.episodes_done.sum()) > 0


def test_kernels_interleave_coherently(gpu, oracle_mod):
    """The bitboard cache stays current across every kind of call: register-resident steps, staged rollouts,
    staged steps (forced), explicit actions, gen_observe, gen_sample."""
    import torch
    cfg, _ = workloads.config("c2_24x24", n_games=53, max_turns=70, spawn_dmin=4)
    env = gpu.GeneralsEnv(cfg, digest=False)
    o = oracle_mod.Oracle(cfg)
    env.reset()
    o.reset()
    kinds = []
    for it in range(12):
        for _ in range(7):
            env.step()
            o.step()
        kinds.append(env.last_launch_register_resident)
        compare(env, o, digest=False, where=f"it {it} steps")
        env.rollout(9, gpu.OBS_NONE)
        o.rollout(9, oracle_mod.OBS_NONE)
        env.set_generic(False, True)
        env.step()
        o.step()
        kinds.append(env.last_launch_register_resident)
        env.set_generic(False, False)
        a = o.sample()
        assert np.array_equal(env.sample().cpu().numpy(), a)
        env.step(torch.from_numpy(a).to(env.device))
        o.step(a)
        env.observe()
        compare(env, o, fields=STATE_FIELDS + OUT_FIELDS[3:], digest=False, where=f"it {it} end")
    assert kinds[0] and not kinds[1]
    assert int(o.episodes_done.sum()) > 0


def test_stack_cache_of_the_biased_policy_is_never_stale(gpu, oracle_mod):
    """gen_buffers.stack_cache (the largest owned stack the observation pass leaves for the next turn's biased
    sampler, R25): the actions drawn must equal the oracle's through everything that invalidates the cache -- resets,
    fused rollouts, staged-kernel steps, explicit-action steps, gen_set_global_step -- and with the cache poisoned by
    hand; a handle without the buffer (the sampler scans the army plane) must agree too."""
    import torch
    cfg, _ = workloads.config("c4_curriculum", n_games=77, max_turns=60)
    env = gpu.GeneralsEnv(cfg, digest=False)
    bare = gpu.GeneralsEnv(cfg, digest=False, stack_cache=False)
    o = oracle_mod.Oracle(cfg)
    for e in (env, bare):
        e.reset()
    o.reset()

    def steps(n, where):
        for t in range(n):
            acts = o.step(want_actions=True)
            for e in (env, bare):
                e.step()
                assert np.array_equal(e.field("actions_out"), acts), f"{where} step {t}"
        compare(env, o, digest=False, where=where)
        compare(bare, o, digest=False, where=where + " (no cache)")

    steps(70, "plain")
    assert int(o.episodes_done.sum()) > 0                       # auto-resets regenerate boards under the cache
    assert env.last_launch_specialised and env.last_launch_register_resident
    assert int((env.tensors["stack_cache"][:, 2] == env.global_step).sum()) == 77      # every stamp is current
    for e in (env, bare):
        e.rollout(5, gpu.OBS_NONE)
    o.rollout(5, oracle_mod.OBS_NONE)
    steps(7, "after a rollout")
    env.set_generic(False, True)                               # one staged-kernel step: the cache goes stale
    acts = o.step(want_actions=True)
    env.step()
    bare.step()
    env.set_generic(False, False)
    steps(9, "after a staged step")
    a = o.sample()
    for e in (env, bare):
        e.step(torch.from_numpy(a).to(e.device))
    o.step(a)
    steps(9, "after explicit actions")
    env.tensors["stack_cache"][:, :2] = 0x7FFFFFF                # wrong stacks under a CURRENT stamp would be used ...
    env.tensors["stack_cache"][:, 2] = 0                         # ... so the stamp is made stale with them
    steps(9, "poisoned cache, stale stamp")
    for e in (env, bare):
        e.reset()
    o.reset()
    steps(30, "after reset")


def test_stack_cache_validity_is_the_handles_knowledge(gpu, oracle_mod):
    """the stamp in gen_buffers.stack_cache can match by accident -- gen_reset puts global_step back to 0,
    explicit-action steps and gen_observe write no stamp, a zeroed cache reads "step 0, owns nothing".  The handle now
    vouches for the cache (previous launch = a BIAS step on this buffer, one step ago); three orders that used to
    sample from a stale cache must give the oracle's actions."""
    import torch
    cfg, _ = workloads.config("c4_curriculum", n_games=77, max_turns=0, auto_reset=0)
    env = gpu.GeneralsEnv(cfg, digest=False)
    o = oracle_mod.Oracle(cfg)
    env.reset()
    o.reset()

    def sampled(n, where):
        for t in range(n):
            acts = o.step(want_actions=True)
            env.step()
            assert np.array_equal(env.field("actions_out"), acts), f"{where} step {t}"
        compare(env, o, digest=False, where=where)

    # 1. k sampler steps leave stamp k; reset; k explicit steps (no stamp written); the sampler at step k
    k = 12
    sampled(k, "before the reset")
    env.reset()
    o.reset()
    for t in range(k):                 # the sampler's moves with the split flipped (R22; valid whenever the move is, R5):
        a = o.sample()                 # the same boards as before the reset now carry different stacks
        kk = a % 9
        a = np.where(kk == 0, a, np.where(kk % 2 == 1, a + 1, a - 1)).astype(np.int32)
        env.step(torch.from_numpy(a).to(env.device))
        o.step(a)
    assert int((env.tensors["stack_cache"][:, 2] == env.global_step).sum()) == 77      # every stale stamp matches
    sampled(6, "reset, explicit steps, sampler")
    # 2. a BIAS step, then the caller rewrites the planes and calls gen_observe (R40)
    gc = np.asarray(o.general_cell)
    for g in range(77):
        for p in range(2):
            if gc[g, p] >= 0:
                o.army[g, gc[g, p]] += 500 + 10 * p
    env.tensors["army"].copy_(torch.from_numpy(np.asarray(o.army).copy()).to(env.device))
    env.observe()
    o.observe()
    sampled(6, "edited planes + gen_observe")
    # 3. a fresh handle, zeroed cache, global step 0, a state written by the caller
    env3 = gpu.GeneralsEnv(cfg, digest=False)
    o3 = oracle_mod.Oracle(cfg)
    env3.reset()
    o3.reset()
    for f in ("army", "owner", "terrain", "turn", "alive", "general_cell"):
        np.asarray(getattr(o3, f))[...] = np.asarray(getattr(o, f))
    o3.observe()
    env3.tensors["stack_cache"].zero_()
    put_board(env3, o3)
    env3.global_step = 0
    assert o3.global_step == 0
    for t in range(4):
        acts = o3.step(want_actions=True)
        env3.step()
        assert np.array_equal(env3.field("actions_out"), acts), f"zeroed cache at step 0: step {t}"
    assert env3.last_launch_register_resident and env3.last_launch_specialised
    compare(env3, o3, digest=False, where="zeroed cache at step 0")


def test_specialised_rollout_kernel_matches_oracle(gpu, oracle_mod):
    cfg, _ = workloads.config("c2_24x24", n_games=70, max_turns=90)
    env, o = make_pair(gpu, oracle_mod, cfg)
    env.reset()
    o.reset()
    for it in range(4):
        env.rollout(32, gpu.OBS_DIGEST)
        o.rollout(32)
        compare(env, o, where=f"rollout {it}")
    assert env.last_launch_specialised


# ------------------------------------------------------------------------------- packed observation (R33)
PACKED_FIELDS = STATE_FIELDS + ["reward", "done", "winner", "obs_army", "obs_packed"]


@pytest.mark.parametrize("name,N,T,over", [
    ("c2_24x24", 90, 200, dict(max_turns=90)),
    ("c5a_2v2", 30, 160, dict(max_turns=100)),
    ("c5b_ffa8", 21, 120, dict(height=12, width=13, n_players=5, spawn_dmin=4, n_cities=4, max_turns=80)),
])
def test_packed_observation_matches_oracle(gpu, oracle_mod, name, N, T, over):
    """The 3-byte-per-cell format (army + one packed byte, R33) on the register-resident kernel and on the staged
    kernel, every step; the three byte planes are not allocated at all."""
    cfg, _ = workloads.config(name, n_games=N, **over)
    env = gpu.GeneralsEnv(cfg, digest=False, packed=True)
    env.set_generic(False, -1)                              # the step kernel also for more than 4 players
    stg = gpu.GeneralsEnv(cfg, digest=True, packed=True, bitboards=False)
    o = oracle_mod.Oracle(cfg)
    for e in (env, stg):
        assert "obs_owner" not in e.tensors and "obs_vis" not in e.tensors
        e.reset()
    o.reset()
    compare(env, o, fields=PACKED_FIELDS, digest=False, where="reset")
    for t in range(T):
        env.step()
        stg.step()
        o.step()
        compare(env, o, fields=PACKED_FIELDS, digest=False, where=f"{name} packed step {t}")
        if t % 8 == 0:
            compare(stg, o, fields=PACKED_FIELDS, digest=True, where=f"{name} packed staged step {t}")
    assert env.last_launch_register_resident and not stg.last_launch_register_resident
    assert int(o.episodes_done.sum()) > 0


def test_packed_rollout_every_step_slots(gpu, oracle_mod):
    K = 6
    cfg, _ = workloads.config("c2_24x24", n_games=41, max_turns=25)
    env = gpu.GeneralsEnv(cfg, k_slots=K, packed=True)
    o = oracle_mod.Oracle(cfg, every_step_K=K)
    env.reset()
    o.reset()
    for it in range(4):
        env.rollout(K, gpu.OBS_EVERY_STEP)
        o.rollout(K, oracle_mod.OBS_EVERY_STEP)
        for k in range(K):
            compare(env, o, fields=["reward", "done", "winner", "obs_army", "obs_packed"], digest=False, slot=k, oslot=k,
                    where=f"it {it} slot {k}")
        compare(env, o, fields=STATE_FIELDS, where=f"it {it}")


# ------------------------------------------------------------------------------- scoreboard history (R34)
@pytest.mark.parametrize("name,N,over", [
    ("c2_24x24", 45, dict(max_turns=70, spawn_dmin=4)),
    ("c5a_2v2", 18, dict(max_turns=60)),
])
def test_scoreboard_history_ring_matches_oracle(gpu, oracle_mod, name, N, over):
    """The 512-slot ring of (land, army_total) per player and turn (R34, the raw material of the paper's temporal
    tokens) written by the step kernel, the staged kernel and fused rollouts, across auto-resets and a ring wrap."""
    cfg, _ = workloads.config(name, n_games=N, **over)
    env = gpu.GeneralsEnv(cfg, digest=False, history=True)
    stg = gpu.GeneralsEnv(cfg, digest=True, history=True, bitboards=False)
    o = oracle_mod.Oracle(cfg)
    for e in (env, stg):
        e.reset()
    o.reset()
    fields = ["score_hist", "land", "army_total", "turn", "episode"]
    compare(env, o, fields=fields, digest=False, where="reset")
    for it in range(8):
        for _ in range(20):
            env.step()
            stg.step()
            o.step()
        compare(env, o, fields=fields, digest=False, where=f"steps {it}")
        compare(stg, o, fields=fields, digest=False, where=f"staged steps {it}")
        for e in (env, stg):
            e.rollout(17, gpu.OBS_NONE)
        o.rollout(17, oracle_mod.OBS_NONE)
        compare(env, o, fields=fields, digest=False, where=f"rollout {it}")
        compare(stg, o, fields=fields, digest=False, where=f"staged rollout {it}")
    assert int(o.episodes_done.sum()) > N                    # several episodes per game
    # ring wrap: one long episode
    cfg2, _ = workloads.config(name, n_games=5, auto_reset=0, max_turns=0, pass_thr=workloads.thr(90))
    env2 = gpu.GeneralsEnv(cfg2, digest=False, history=True)
    o2 = oracle_mod.Oracle(cfg2)
    env2.reset()
    o2.reset()
    for _ in range(19):
        env2.rollout(32, gpu.OBS_NONE)
        o2.rollout(32, oracle_mod.OBS_NONE)
    env2.step()
    o2.step()
    assert int(o2.turn.max()) > 512
    compare(env2, o2, fields=fields, digest=False, where="wrap")


# ------------------------------------------------------------------------------- rollout == steps
@pytest.mark.parametrize("mode", ["digest", "none"])
def test_rollout_equals_steps(gpu, oracle_mod, mode):
    cfg, _ = workloads.config("c2_24x24", n_games=70, max_turns=90)
    env, o = make_pair(gpu, oracle_mod, cfg)
    env.reset()
    o.reset()
    K = 32
    for it in range(5):
        env.rollout(K, gpu.OBS_DIGEST if mode == "digest" else gpu.OBS_NONE)
        o.rollout(K)
        if mode == "digest":
            compare(env, o, where=f"rollout {it}")
        else:
            compare(env, o, fields=STATE_FIELDS + ["reward", "done", "winner"], digest=False, where=f"rollout {it}")
    assert env.global_step == 5 * K


def test_rollout_every_step_slots(gpu, oracle_mod):
    K = 12
    cfg, _ = workloads.config("c2_24x24", n_games=37, max_turns=20)
    env, o = make_pair(gpu, oracle_mod, cfg, k_slots=K)
    env.reset()
    o.reset()
    for it in range(3):
        env.rollout(K, gpu.OBS_EVERY_STEP)
        o.rollout(K, oracle_mod.OBS_EVERY_STEP)
        env.torch.cuda.synchronize()
        for k in range(K):
            compare(env, o, fields=OUT_FIELDS, digest=False, slot=k, oslot=k, where=f"it {it} slot {k}")
        compare(env, o, fields=STATE_FIELDS, where=f"it {it}")


def test_K_split_and_batch_split_independence(gpu, oracle_mod):
    """M2: rollout(48) == rollout(16) x 3 == 48 steps; a game_id_base split reproduces the same games."""
    cfg, _ = workloads.config("c2_24x24", n_games=50, max_turns=40)
    a = gpu.GeneralsEnv(cfg)
    a.reset()
    a.rollout(48)
    b = gpu.GeneralsEnv(cfg)
    b.reset()
    for _ in range(3):
        b.rollout(16)
    c0 = gpu.GeneralsEnv(dict(cfg, n_games=19))
    c1 = gpu.GeneralsEnv(dict(cfg, n_games=31, game_id_base=19))
    for c in (c0, c1):
        c.set_launch(4)
        c.reset()
        for _ in range(48):
            c.step()
    for f in STATE_FIELDS + ["obs_digest", "obs_army", "obs_owner", "obs_terrain", "obs_vis", "reward", "done"]:
        assert np.array_equal(a.field(f), b.field(f)), f
        assert np.array_equal(a.field(f), np.concatenate([c0.field(f), c1.field(f)], axis=0)), f


@pytest.mark.parametrize("wpc", [4, 8, 16, 32])
def test_launch_geometry_does_not_change_results(gpu, oracle_mod, wpc):
    cfg, _ = workloads.config("c1_8x8", n_games=45, auto_reset=1, max_turns=50)
    env, o = make_pair(gpu, oracle_mod, cfg)
    env.set_launch(wpc)
    env.reset()
    o.reset()
    for _ in range(4):
        env.rollout(30)
        o.rollout(30)
    compare(env, o, where=f"wpc {wpc}")


# ------------------------------------------------------------------------------- hand-built boards
def dict_(a, b):
    d = dict(a)
    d.update(b)
    return d


def put_board(env, o):
    """Copy a hand-built oracle state into the device buffers and let the library observe it."""
    import torch
    for f in ("army", "owner", "terrain", "turn", "alive", "general_cell", "done", "winner"):
        src = np.asarray(getattr(o, f))
        if f in ("done", "winner"):
            src = src[0]
        env.tensors[f].view(-1).copy_(torch.from_numpy(src.reshape(-1).copy()).to(env.device))
    env.observe()


def run_hand_case(gpu, oracle_mod, H, W, P, cells, actions, turn=0, team_size=1, steps=1, **cfg):
    import torch
    from helpers import hand_board
    o = hand_board(oracle_mod, H, W, P, cells, turn=turn, team_size=team_size, **cfg)
    base = dict(n_games=1, height=H, width=W, n_players=P, team_size=team_size)
    base.update(cfg)
    env = gpu.GeneralsEnv(base, digest=False)                      # register-resident step kernel
    twin = gpu.GeneralsEnv(base, digest=False, bitboards=False)    # staged kernel
    for e in (env, twin):
        put_board(e, o)
        compare(e, o, fields=["land", "army_total"] + OUT_FIELDS[3:], digest=False, where="observe")
    for s in range(steps):
        a = np.asarray(actions[s] if steps > 1 else actions, dtype=np.int32).reshape(1, P)
        o.step(a)
        for e in (env, twin):
            e.step(torch.from_numpy(a).to(e.device))
            compare(e, o, digest=False, where=f"hand step {s}")
    assert env.last_launch_register_resident and not twin.last_launch_register_resident
    return env, o


W8_CELLS = {(0, 0): (GN, 0, 3), (3, 2): (PL, 0, 10), (3, 3): (GN, 1, 4), (2, 3): (PL, 1, 7),
            (1, 3): (PL, 1, 1), (2, 2): (PL, 1, 2), (0, 3): (CT, -1, 45), (1, 1): (MT, -1, 0)}


@pytest.mark.parametrize("flags", [0, 2])
def test_W8_capture_on_gpu(gpu, oracle_mod, flags):
    env, o = run_hand_case(gpu, oracle_mod, 4, 4, 2, W8_CELLS, [act(3, 2, 4, RIGHT), act(2, 3, 4, LEFT)],
                           turn=10, rule_flags=flags)
    assert env.field("army_total")[0].tolist() == [13 if flags else 15, 0]     # the paper-derived value
    assert env.field("reward")[0].tolist() == [1, -1] and int(env.field("done")[0]) == 1


def test_hand_cases_on_gpu(gpu, oracle_mod):
    g2 = {(0, 0): (GN, 0, 1), (2, 2): (GN, 1, 1)}
    # W1, W3, W4 (three outcomes), W5 (castle), W6 / W7 (simultaneous), W11 (saturation)
    cases = [
        (dict_(g2, {(1, 0): (PL, 0, 5)}), [act(1, 0, 3, RIGHT), PASS]),
        (dict_(g2, {(1, 0): (PL, 0, 5), (1, 1): (PL, 0, 3)}), [act(1, 0, 3, RIGHT), PASS]),
        (dict_(g2, {(1, 0): (PL, 0, 5), (1, 1): (PL, 1, 3)}), [act(1, 0, 3, RIGHT), PASS]),
        (dict_(g2, {(1, 0): (PL, 0, 5), (1, 1): (PL, 1, 4)}), [act(1, 0, 3, RIGHT), PASS]),
        (dict_(g2, {(1, 0): (PL, 0, 5), (1, 1): (PL, 1, 7)}), [act(1, 0, 3, RIGHT), PASS]),
        (dict_(g2, {(1, 0): (PL, 0, 51), (1, 1): (CT, -1, 45)}), [act(1, 0, 3, RIGHT), PASS]),
        (dict_(g2, {(1, 0): (PL, 0, 46), (1, 1): (CT, -1, 45)}), [act(1, 0, 3, RIGHT), PASS]),
        (dict_(g2, {(1, 0): (PL, 0, 4), (1, 2): (PL, 1, 6)}), [act(1, 0, 3, RIGHT), act(1, 2, 3, LEFT)]),
        (dict_(g2, {(1, 0): (PL, 0, 5), (1, 1): (PL, 1, 5)}), [act(1, 0, 3, RIGHT), act(1, 1, 3, LEFT)]),
        (dict_(g2, {(1, 0): (PL, 0, 21), (1, 1): (PL, 0, 32760)}), [act(1, 0, 3, RIGHT), PASS]),
        (dict_(g2, {(1, 0): (PL, 0, 7)}), [act(1, 0, 3, RIGHT, half=1), PASS]),
        (dict_(g2, {(1, 1): (PL, 0, 5), (0, 1): (MT, -1, 0)}), [act(1, 1, 3, UP), PASS]),
        (dict_(g2, {(1, 1): (PL, 0, 5)}), [act(1, 1, 3, DOWN), act(2, 2, 3, UP)]),
    ]
    for cells, a in cases:
        for turn in (0, 1, 49, 99):
            run_hand_case(gpu, oracle_mod, 3, 3, 2, cells, a, turn=turn)
            run_hand_case(gpu, oracle_mod, 3, 3, 2, cells, a, turn=turn, rule_flags=4)
    env, _ = run_hand_case(gpu, oracle_mod, 3, 3, 2, cases[9][0], cases[9][1])
    assert int(env.field("sat_events")[0]) == 1


def test_W13_unclaimed_general_on_gpu(gpu, oracle_mod):
    """R40: gen_observe turns a GENERAL cell that is nobody's recorded general into a CITY (the raw planes are written
    to the device un-normalised); afterwards both step kernels play W13 like the oracle."""
    import torch
    from helpers import hand_board
    cells = {(0, 0): (GN, 0, 5), (2, 2): (GN, 1, 3), (0, 1): (GN, -1, 2), (2, 0): (GN, 1, 1), (1, 0): (PL, 0, 6)}
    seq = [[act(0, 0, 3, RIGHT), PASS], [act(1, 0, 3, DOWN), PASS]]
    for bitboards in (True, False):
        o = hand_board(oracle_mod, 3, 3, 2, cells, turn=0)
        env = gpu.GeneralsEnv(dict(n_games=1, height=3, width=3, n_players=2, team_size=1), digest=False, bitboards=bitboards)
        put_board(env, o)
        raw = env.tensors["terrain"].clone()
        raw[0, 1] = GN
        raw[0, 6] = GN
        env.tensors["terrain"].copy_(raw)
        env.observe()
        compare(env, o, digest=False, where="W13 observe")
        assert env.field("terrain")[0, 1] == CT and env.field("terrain")[0, 6] == CT
        for a in seq:
            a = np.asarray(a, dtype=np.int32).reshape(1, 2)
            o.step(a)
            env.step(torch.from_numpy(a).to(env.device))
            compare(env, o, digest=False, where="W13 step")
        assert env.last_launch_register_resident == bitboards
        assert int(env.field("alive")[0]) == 0b11 and env.field("land")[0].tolist() == [4, 1]


def test_saturating_growth_on_gpu(gpu, oracle_mod):
    cells = {(0, 0): (GN, 0, 32766), (2, 2): (GN, 1, 1), (1, 1): (CT, 0, 32767), (0, 1): (PL, 0, 32767)}
    seq = [[PASS, PASS]] * 4
    env, o = run_hand_case(gpu, oracle_mod, 3, 3, 2, cells, seq, turn=47, steps=4)
    assert int(env.field("sat_events")[0]) == int(o.sat_events[0]) > 0


def test_team_rules_on_gpu(gpu, oracle_mod):
    base = {(0, 0): (GN, 0, 1), (0, 4): (GN, 2, 1), (4, 0): (GN, 3, 1), (2, 0): (PL, 0, 6)}
    run_hand_case(gpu, oracle_mod, 5, 5, 4, dict_(base, {(2, 1): (PL, 1, 3), (4, 4): (GN, 1, 1)}),
                  [act(2, 0, 5, RIGHT), PASS, PASS, PASS], team_size=2)
    run_hand_case(gpu, oracle_mod, 5, 5, 4, dict_(base, {(2, 1): (GN, 1, 3)}),
                  [act(2, 0, 5, RIGHT), PASS, PASS, PASS], team_size=2)
    cells = {(0, 0): (GN, 0, 1), (0, 2): (GN, 2, 1), (0, 1): (PL, 0, 9), (2, 2): (GN, 3, 1),
             (2, 1): (PL, 1, 9), (2, 0): (GN, 1, 1), (1, 2): (PL, 3, 4)}
    env, o = run_hand_case(gpu, oracle_mod, 3, 3, 4, cells,
                           [[act(0, 1, 3, RIGHT), PASS, PASS, PASS], [PASS, act(2, 1, 3, RIGHT), PASS, PASS]],
                           team_size=2, steps=2)
    assert env.field("reward")[0].tolist() == [1, 1, -1, -1]


def test_B3_exhaustive_joint_actions_3x3(gpu, oracle_mod):
    """B3: every joint action pair (81 x 81) on a 3x3 board, one game per pair, in one batch."""
    import torch
    from helpers import hand_board
    cells = {(0, 0): (GN, 0, 4), (2, 2): (GN, 1, 3), (0, 1): (PL, 0, 3), (1, 1): (PL, 1, 5),
             (1, 0): (CT, -1, 2), (2, 0): (MT, -1, 0), (1, 2): (PL, 1, 2), (0, 2): (PL, 0, 2)}
    one = hand_board(oracle_mod, 3, 3, 2, cells, turn=1)
    N = 81 * 81
    cfg = dict(n_games=N, height=3, width=3, n_players=2)
    o = oracle_mod.Oracle(cfg)
    for f in ("army", "owner", "terrain", "turn", "alive", "general_cell"):
        getattr(o, f)[...] = getattr(one, f)[0]
    o.winner[:] = -1
    o.observe()
    env = gpu.GeneralsEnv(cfg, digest=False)
    put_board(env, o)
    a = np.stack(np.meshgrid(np.arange(81), np.arange(81), indexing="ij"), -1).reshape(N, 2).astype(np.int32)
    env.step(torch.from_numpy(a).to(env.device))
    o.step(a)
    compare(env, o, digest=False, where="B3")
    assert len({bytes(x) for x in env.field("army")}) > 30      # many distinct outcomes


def test_frozen_games_and_empty_batch(gpu, oracle_mod):
    cfg, _ = workloads.config("c1_8x8", n_games=30, max_turns=12, auto_reset=0)
    env, o = make_pair(gpu, oracle_mod, cfg)
    env.reset()
    o.reset()
    for t in range(20):
        env.step()
        o.step()
        compare(env, o, where=f"frozen {t}")
    assert (env.field("done") == 2).all() and (env.field("turn") == 12).all()
    env.rollout(5)
    o.rollout(5)
    compare(env, o, where="frozen rollout")
    # explicit actions on frozen games (R31): nothing is applied and actions_out reports 0, on both step kernels
    import torch
    rng = np.random.default_rng(11)
    for staged in (False, True):
        e2 = gpu.GeneralsEnv(cfg, digest=staged)
        o2 = oracle_mod.Oracle(cfg)
        e2.reset()
        o2.reset()
        for t in range(16):
            a = workloads.random_actions(rng, 30, 2, 8, 8) if t % 2 else o2.sample()
            e2.step(torch.from_numpy(a).to(e2.device))
            want = o2.step(a, want_actions=True)
            compare(e2, o2, digest=staged, where=f"frozen explicit {t}")
            assert np.array_equal(e2.field("actions_out"), want), t
        assert (e2.field("done") == 2).all() and (e2.field("actions_out") == 0).all()
        assert e2.last_launch_register_resident == (not staged)
    empty = gpu.GeneralsEnv(dict(cfg, n_games=0))
    empty.reset()
    empty.step()
    empty.rollout(3)
    assert empty.launch_count == 0


def test_sample_only_matches_oracle(gpu, oracle_mod):
    cfg, _ = workloads.config("c4_curriculum", n_games=64, height=12, width=12, spawn_dmax=9, n_cities=4)
    env, o = make_pair(gpu, oracle_mod, cfg)
    env.reset()
    o.reset()
    for t in range(60):
        got = env.sample().cpu().numpy()
        assert np.array_equal(got, o.sample()), t
        env.step()
        o.step()


def test_keep_episode_reset(gpu, oracle_mod):
    import torch
    cfg, _ = workloads.config("c1_8x8", n_games=16)
    env = gpu.GeneralsEnv(cfg)
    env.reset()
    first = env.field("terrain").copy()
    env.tensors["episode"].copy_(torch.arange(16, dtype=torch.int32, device=env.device))
    env.reset(keep_episode=True)
    again = env.field("terrain")
    assert np.array_equal(again[0], first[0]) and not np.array_equal(again[1:], first[1:])
    assert env.field("episode").tolist() == list(range(16))


@pytest.mark.parametrize("pinned,N", [(True, 32), (False, 32), (True, 37), (True, 3000)])
def test_step_host_end_to_end(gpu, oracle_mod, pinned, N):
    """gen_step_host: pinned host buffers are used in place (the step kernel reads the actions through their device
    alias, one small kernel writes reward + done into the host arrays); pageable buffers take the memcpy route; odd
    sizes exercise the unaligned tails.  Mixed: pinned actions with pageable results and the other way round."""
    import torch
    cfg, _ = workloads.config("c1_8x8", n_games=N, auto_reset=1, max_turns=30)
    env, o = make_pair(gpu, oracle_mod, cfg)
    env.reset()
    o.reset()
    mk = (lambda t: t.pin_memory()) if pinned else (lambda t: t)
    h_a = mk(torch.zeros((N, 2), dtype=torch.int32))
    h_r = mk(torch.zeros((N, 2), dtype=torch.int8))
    h_d = mk(torch.zeros((N,), dtype=torch.uint8))
    h_r2 = torch.zeros((N, 2), dtype=torch.int8)                 # pageable
    h_a2 = torch.zeros((N, 2), dtype=torch.int32).pin_memory()  # pinned
    for t in range(60):
        a = o.sample()
        if t % 3 == 2:                                           # mixed kinds of memory in one call
            h_a2.copy_(torch.from_numpy(a))
            env.step_host(h_a2, h_r2, h_d)
            o.step(a)
            assert np.array_equal(h_r2.numpy(), o.reward[0]) and np.array_equal(h_d.numpy(), o.done[0])
            continue
        h_a.copy_(torch.from_numpy(a))
        env.step_host(h_a, h_r, h_d)
        o.step(a)
        assert np.array_equal(h_r.numpy(), o.reward[0]) and np.array_equal(h_d.numpy(), o.done[0])
    env.step_host(None, None, h_d)                               # sampler, done only
    o.step()
    assert np.array_equal(h_d.numpy(), o.done[0])
    compare(env, o, where="step_host")
    assert int(o.episodes_done.sum()) > 0


def test_step_host_with_an_odd_reward_pointer(gpu, oracle_mod):
    """a pinned int8 result array that starts at an odd address (a slice of a byte buffer).  The step
    kernel's own host write of a two-player reward row is one 16-bit store; such an array must take the byte-wise
    mirror kernel instead of faulting."""
    import torch
    N = 203
    cfg, _ = workloads.config("c2_24x24", n_games=N, max_turns=25)
    env = gpu.GeneralsEnv(cfg, digest=False)
    o = oracle_mod.Oracle(cfg)
    env.reset()
    o.reset()
    raw = torch.zeros(2 * N + 1, dtype=torch.int8).pin_memory()
    h_r = raw[1:]
    assert h_r.data_ptr() % 2 == 1 and h_r.is_contiguous()
    h_d = torch.zeros((N,), dtype=torch.uint8).pin_memory()
    for t in range(40):
        before = env.launch_count
        if t % 2:
            env.step_host(None, h_r, h_d)
        else:
            env.step_host_async(None, h_r, h_d)
            env.host_wait(0)
        o.step()
        assert env.launch_count == before + 2                     # the step and the mirror kernel
        assert np.array_equal(h_r.numpy().reshape(N, 2), o.reward[0]) and np.array_equal(h_d.numpy(), o.done[0])
    assert env.last_launch_register_resident and int(o.episodes_done.sum()) > 0
    compare(env, o, digest=False, where="odd reward pointer")


def test_step_host_async_more_than_four_calls_and_many_action_arrays(gpu, oracle_mod):
    """(a) "at most 4 calls in flight" is now kept by the library -- six calls issued with no wait in
    between (six sets of host slots), then one wait: every call's results are in its own slots; (b) a new pinned
    actions array every step (twelve of them in rotation) next to one fixed pair of result arrays."""
    import torch
    N = 203
    cfg, _ = workloads.config("c2_24x24", n_games=N, max_turns=30)
    env = gpu.GeneralsEnv(cfg, digest=False)
    o = oracle_mod.Oracle(cfg)
    env.reset()
    o.reset()
    slots = [dict(r=torch.full((N, 2), 99, dtype=torch.int8).pin_memory(),
                  d=torch.full((N,), 99, dtype=torch.uint8).pin_memory()) for _ in range(6)]
    for rnd in range(6):
        want = []
        for s in slots:
            env.step_host_async(None, s["r"], s["d"])            # no wait: the fifth and sixth call wait inside
            o.step()
            want.append((o.reward[0].copy(), o.done[0].copy()))
        env.host_wait(0)
        for i, s in enumerate(slots):
            assert np.array_equal(s["r"].numpy(), want[i][0]) and np.array_equal(s["d"].numpy(), want[i][1]), (rnd, i)
    many = [torch.zeros((N, 2), dtype=torch.int32).pin_memory() for _ in range(12)]
    h_r, h_d = slots[0]["r"], slots[0]["d"]
    for t in range(36):
        a = o.sample()
        many[t % 12].copy_(torch.from_numpy(a))
        env.step_host(many[t % 12], h_r, h_d)
        o.step(a)
        assert np.array_equal(h_r.numpy(), o.reward[0]) and np.array_equal(h_d.numpy(), o.done[0]), t
    compare(env, o, digest=False, where="async in-flight limit / many action arrays")
    assert int(o.episodes_done.sum()) > 0


def test_checkpoint_and_resume(gpu, oracle_mod):
    """SURVEY section 5 (checkpoint / resume): the handle holds no game state -- everything lives in the caller's
    tensors plus the global step -- so cloning the STATE tensors and gen_global_step is a checkpoint.  A fresh handle
    that is given the cloned state (derived caches rebuilt by gen_observe, nothing else copied) must continue bit for
    bit like the original and like the oracle, through auto-resets, on the per-step kernel and through a fused
    rollout."""
    cfg, _ = workloads.config("c4_curriculum", n_games=150, max_turns=45)
    env = gpu.GeneralsEnv(cfg, digest=False, history=True)
    o = oracle_mod.Oracle(cfg)
    env.reset()
    o.reset()
    for _ in range(60):
        env.step()
        o.step()
    state = ["army", "owner", "terrain", "turn", "episode", "alive", "general_cell", "done", "winner", "episodes_done",
             "wins", "truncations", "sat_events", "invalid_actions", "play_size", "score_hist"]
    ckpt = {k: env.tensors[k].clone() for k in state}
    step0 = env.global_step
    twin = gpu.GeneralsEnv(cfg, digest=False, history=True)    # nothing but the checkpoint goes in
    for k in state:
        twin.tensors[k].copy_(ckpt[k])
    twin.global_step = step0
    twin.observe()                                              # scoreboard, bitboard cache and observation from the planes
    for t in range(70):
        env.step()
        twin.step()
        o.step()
        if t % 10 == 9:
            compare(env, o, digest=False, where=f"original, step {t}")
            compare(twin, o, digest=False, where=f"resumed, step {t}")
    assert np.array_equal(twin.field("score_hist"), env.field("score_hist"))
    for e in (env, twin):
        e.rollout(9, gpu.OBS_NONE)
    o.rollout(9, oracle_mod.OBS_NONE)
    compare(twin, o, fields=STATE_FIELDS, digest=False, where="resumed, after a rollout")
    assert twin.last_launch_register_resident is False and int(o.episodes_done.sum()) > 100


def test_actions_produced_on_the_device_between_chained_steps(gpu, oracle_mod):
    """a chained gen_step skips the grid-wide wait, so it must never be chained when it consumes actions
    another kernel produced.  Here a foreign kernel (a torch elementwise op) writes the actions into ONE reused
    buffer right before every explicit-action step, sampler steps (which do chain) run in between, nothing
    synchronises the stream: a step that started before its producer had finished would read the previous turn's
    actions and diverge from the oracle."""
    import torch
    N, T = 2048, 36
    cfg, _ = workloads.config("c2_24x24", n_games=N, max_turns=30)
    env = gpu.GeneralsEnv(cfg, digest=False)
    o = oracle_mod.Oracle(cfg)
    env.reset()
    o.reset()
    explicit = [t % 3 != 2 for t in range(T)]
    stream = []                                               # the oracle plays first: its sampled actions are the inputs
    for t in range(T):
        if explicit[t]:
            a = o.sample()
            stream.append(a)
            o.step(a)
        else:
            stream.append(None)
            o.step()
    dev_all = torch.from_numpy(np.stack([a if a is not None else np.zeros((N, 2), np.int32) for a in stream])).to(env.device)
    acts = torch.zeros((N, 2), dtype=torch.int32, device=env.device)
    zero = torch.zeros((N, 2), dtype=torch.int32, device=env.device)
    torch.cuda.synchronize()
    for t in range(T):
        if explicit[t]:
            torch.add(dev_all[t], zero, out=acts)             # the producer: same buffer every time
            env.step(acts)
        else:
            env.step()                                        # built-in sampler: these launches chain
    compare(env, o, digest=False, where="device-produced actions between chained steps")
    assert env.last_launch_register_resident and int(o.episodes_done.sum()) > 0


@pytest.mark.parametrize("name,N,over", [
    ("c2_24x24", 203, dict(max_turns=40)),
    ("c5a_2v2", 37, dict(height=12, width=12, n_cities=3, spawn_dmin=4, max_turns=30)),     # P = 4: byte-wise reward writes
    ("c5b_ffa8", 21, dict(height=12, width=13, n_players=3, spawn_dmin=4, n_cities=4, max_turns=30)),
])
def test_step_host_async_one_step_late(gpu, oracle_mod, name, N, over):
    """gen_step_host_async + gen_host_wait: the loop the end-to-end bench leg times -- two sets of pinned host slots,
    step t issued before the results of step t - 1 are read (lag 1), then the last one drained (lag 0); results of
    every step equal the oracle's, state equal at the end; forgetting the alias table in between changes nothing.
    The step kernel writes reward + done to the host arrays itself (2, 3 and 4 players: the reward row is written
    as one halfword or byte by byte)."""
    import torch
    cfg, _ = workloads.config(name, n_games=N, **over)
    P = cfg["n_players"]
    env = gpu.GeneralsEnv(cfg, digest=False)
    o = oracle_mod.Oracle(cfg)
    env.reset()
    o.reset()
    slots = [dict(a=torch.zeros((N, P), dtype=torch.int32).pin_memory(), r=torch.full((N, P), 99, dtype=torch.int8).pin_memory(),
                  d=torch.full((N,), 99, dtype=torch.uint8).pin_memory()) for _ in range(2)]
    want = []
    T = 90
    for t in range(T):
        s = slots[t & 1]
        a = o.sample()
        s["a"].copy_(torch.from_numpy(a))
        env.step_host_async(s["a"], s["r"], s["d"])
        o.step(a)
        want.append((o.reward[0].copy(), o.done[0].copy()))
        if t >= 1:
            env.host_wait(1)                                     # step t - 1 has landed; step t may still run
            p = slots[(t - 1) & 1]
            assert np.array_equal(p["r"].numpy(), want[t - 1][0]) and np.array_equal(p["d"].numpy(), want[t - 1][1]), t
        if t == 40:
            env.forget_host_buffers()
    env.host_wait(0)
    p = slots[(T - 1) & 1]
    assert np.array_equal(p["r"].numpy(), want[-1][0]) and np.array_equal(p["d"].numpy(), want[-1][1])
    compare(env, o, digest=False, where="step_host_async")
    assert env.last_launch_register_resident and int(o.episodes_done.sum()) > 0
    n_before = env.launch_count
    env.step_host_async(None, slots[0]["r"], slots[0]["d"])       # sampler + host results: still one launch (no mirror kernel)
    env.host_wait(0)
    o.step()
    assert env.launch_count == n_before + 1
    assert np.array_equal(slots[0]["r"].numpy(), o.reward[0]) and np.array_equal(slots[0]["d"].numpy(), o.done[0])
    with pytest.raises(gpu.GenError):
        env.host_wait(4)


# ------------------------------------------------------------------------------- full-size sampled check
@pytest.mark.parametrize("digest", [False, True])
def test_config2_full_size_sampled_games(gpu, oracle_mod, digest):
    """BASELINE config 2 at its full N = 16,384 in the launch configuration bench.py times (digest False:
    the register-resident step kernel; True: the staged kernel with the digest chained): the oracle
    replays a sample of global game ids (first / last / strided; legitimate because a game depends on
    its global id only, M2) and must agree on state, observation and digest."""
    cfg, _ = workloads.config("c2_24x24")
    env = gpu.GeneralsEnv(cfg, digest=digest)
    env.reset()
    T = 240
    for _ in range(T):
        env.step()
    env.torch.cuda.synchronize()
    ids = sorted(set(list(range(0, 24)) + list(range(16384 - 24, 16384)) + list(range(5, 16384, 1571))))
    for gid in ids:
        o = oracle_mod.Oracle(dict(cfg, n_games=1, game_id_base=gid))
        o.reset()
        for _ in range(T):
            o.step()
        for f in STATE_FIELDS + OUT_FIELDS:
            got = env.field(f)[gid]
            want = np.asarray(o.field(f))[0]
            assert np.array_equal(got, want), (gid, f)
        if digest:
            assert int(env.field("obs_digest")[gid]) == int(o.obs_digest[0]), gid
    assert env.last_launch_register_resident == (not digest) and env.last_launch_specialised
    # properties that hold at any size
    owner, terrain, army = env.field("owner"), env.field("terrain"), env.field("army")
    assert (owner[terrain == MT] == -1).all() and (army >= 0).all()
    for p in range(2):
        assert np.array_equal(env.field("land")[:, p], (owner[:, :576] == p).sum(1))
        assert np.array_equal(env.field("army_total")[:, p],
                              np.where(owner[:, :576] == p, army[:, :576], 0).astype(np.int64).sum(1))
    vis = env.field("obs_vis")
    assert ((owner[:, None, :] == np.arange(2)[None, :, None]) <= vis.astype(bool)).all()


@pytest.mark.parametrize("name,n_ids,history", [
    ("c2_24x24", 64, True),          # 16,384 games x 2,000 steps
    ("c3_sweep", 32, False),         # 262,144 games x 1,000 steps
    ("c4_curriculum", 24, False),    # 65,536 games x 4,000 steps, biased policy
    ("c5a_2v2", 16, False),          # 32,768 games x 2,000 steps, 2v2 on 32x32
    ("c5b_ffa8", 10, False),         # 32,768 games x 2,000 steps, 8-player free-for-all
])
def test_configs_full_length(gpu, oracle_mod, name, n_ids, history):
    """BASELINE configs 2-5 in full -- every game of the batch stepped for the config's whole length with auto-reset,
    in the launch configuration bench.py times (bitboard cache, no digest, chained launches where they apply).  The
    oracle replays a sample of global game ids over all turns: state, observation and accumulators (episodes
    finished, wins, truncations, saturations) must agree at the end; for config 2 the scoreboard history ring (R34)
    pins the last 512 turns of the trajectory on the way."""
    cfg, T = workloads.config(name)
    N = cfg["n_games"]
    env = gpu.GeneralsEnv(cfg, digest=False, actions_out=False, history=history)
    env.reset()
    for _ in range(T):
        env.step()
    env.torch.cuda.synchronize()
    assert env.global_step == T
    stride = max(1, N // max(1, n_ids - 4))
    ids = sorted(set([0, 1, N - 2, N - 1] + list(range(stride // 2, N, stride))))
    fields = STATE_FIELDS + OUT_FIELDS + (["score_hist"] if history else [])
    import torch
    sel = torch.tensor(ids, device=env.device)
    got = {}
    for f in fields:
        t = env.tensors[f][0] if f in OUT_FIELDS else env.tensors[f]
        got[f] = t.index_select(0, sel).cpu().numpy()
    for k, gid in enumerate(ids):
        o = oracle_mod.Oracle(dict(cfg, n_games=1, game_id_base=gid))
        o.reset()
        for _ in range(T):
            o.step()
        for f in fields:
            want = np.asarray(o.field(f))[0] if f != "score_hist" else np.asarray(o.score_hist)[0]
            have = got[f][k]
            if have.dtype != want.dtype:
                have = have.view(want.dtype)
            assert np.array_equal(have, want.reshape(have.shape)), (name, gid, f)
    assert int(env.tensors["episodes_done"].sum()) > 0


@pytest.mark.parametrize("name,N,T,roll", [
    ("c3_sweep", 262144, 130, 32),        # config 3: steps interleaved with fused rollouts
    ("c3_sweep", 1048576, 70, 0),
    ("c4_curriculum", 65536, 150, 0),     # biased policy (R25): the step kernel scans the army plane for the largest stack
    ("c5a_2v2", 32768, 120, 0),
    ("c5b_ffa8", 32768, 120, 0),
    ("c4_flags", 65536, 150, 0),          # NEXT-4: all three alternative rule readings at scale (uniform policy)
])
def test_full_size_configs_sampled_games(gpu, oracle_mod, name, N, T, roll):
    """BASELINE configs 3, 4, 5 at their full batch sizes, in the launch configuration bench.py --sweep times
    (bitboard cache, no digest buffer): the oracle replays a sample of global game ids one by one (first /
    last / strided: a game depends on its global id only, M2) and must agree on every tensor; plus properties
    that hold at any size."""
    import torch
    if name == "c4_flags":                                   # short spawn distances: captures (floor halving), ticks, rotation
        cfg, _ = workloads.config("c4_curriculum", n_games=N, rule_flags=7, bias_thr=0, spawn_dmax=8, max_turns=120)
    else:
        cfg, _ = workloads.config(name, n_games=N)
    P, HW = cfg["n_players"], cfg["height"] * cfg["width"]
    env = gpu.GeneralsEnv(cfg, digest=False, actions_out=False)
    env.reset()
    plan = []                                                # the same call sequence on both sides
    t = 0
    while t < T:
        if roll and t % 50 == 10:
            env.rollout(roll, gpu.OBS_NONE)
            plan.append(roll)
            t += roll
        else:
            env.step()
            plan.append(1)
            t += 1
    env.step()                                               # a state-only rollout leaves no observation: end on a step
    plan.append(1)
    env.torch.cuda.synchronize()
    ids = sorted(set(list(range(12)) + list(range(N - 12, N)) + list(range(7, N, N // 23))))
    sel = torch.tensor(ids, device=env.device)
    fields = [f for f in STATE_FIELDS + OUT_FIELDS]
    got = {}
    for f in fields:
        tns = env.tensors[f]
        if f in OUT_FIELDS:
            tns = tns[0]
        got[f] = tns.index_select(0, sel).cpu().numpy()
    for k, gid in enumerate(ids):
        o = oracle_mod.Oracle(dict(cfg, n_games=1, game_id_base=gid))
        o.reset()
        for n in plan:
            if n == 1:
                o.step()
            else:
                o.rollout(n, oracle_mod.OBS_NONE)
        for f in fields:
            want = np.asarray(o.field(f))[0]
            have = got[f][k]
            if have.dtype != want.dtype:
                have = have.view(want.dtype)
            assert np.array_equal(have, want.reshape(have.shape)), (name, gid, f)
    # properties that hold at any size (all games)
    owner, army, terrain = env.tensors["owner"][:, :HW], env.tensors["army"][:, :HW], env.tensors["terrain"][:, :HW]
    assert bool((army >= 0).all()) and bool((owner[terrain == MT] == -1).all())
    for p in range(P):
        mine = owner == p
        assert torch.equal(env.tensors["land"][:, p], mine.sum(1).to(torch.int32))
        assert torch.equal(env.tensors["army_total"][:, p].to(torch.int64), (army.to(torch.int64) * mine).sum(1))
        assert bool((env.tensors["obs_vis"][0, :, p, :HW][mine] == 1).all())      # fog: vis contains owned (I5)
    assert int(env.tensors["episodes_done"].sum()) >= 0


def _sample_ids(N, extra=23):
    return sorted(set(list(range(12)) + list(range(N - 12, N)) + list(range(7, N, max(1, N // extra)))))


def _gather(env, fields, ids, slot=0):
    import torch
    sel = torch.tensor(ids, device=env.device)
    out = {}
    for f in fields:
        t = env.tensors[f]
        if f in OUT_FIELDS or f in ("obs_packed", "actions_out"):
            t = t[slot]
        out[f] = t.index_select(0, sel).cpu().numpy()
    return out


def _same_game(have, want, what):
    if have.dtype != want.dtype:
        have = have.view(want.dtype)
    assert np.array_equal(have, want.reshape(have.shape)), what


@pytest.mark.parametrize("leg,N,variant", [
    ("rollout_digest", 16384, 3), ("rollout_digest", 262144, 3),
    ("rollout_every", 16384, 22), ("rollout_every", 262144, 22),
    ("packed", 16384, 7), ("packed", 262144, 7),
    ("host_async", 16384, 7),
])
def test_timed_legs_at_their_own_size_and_mode(gpu, oracle_mod, leg, N, variant):
    """the kernel build that runs is a function of the batch size and of the output format
    (pick_variant), so every leg bench.py publishes is checked here at its own size and in its own mode -- the fused
    32-turn digest rollout, the 8-turn rollout that writes every turn's planes, the packed observation, and the
    end-to-end loop whose step kernel writes reward / done into pinned host arrays -- on BASELINE config 2 / 3's boards
    (max_turns shortened so that auto-resets fall inside the run; it is a run-time parameter, the build is the same).
    The oracle replays a sample of global game ids (first / last / strided: a game depends on its id only)."""
    import torch
    cfg, _ = workloads.config("c2_24x24" if N == 16384 else "c3_sweep", n_games=N, max_turns=70)
    ids = _sample_ids(N, 15)
    lib = gpu.load_library()

    def oracles(**kw):
        out = []
        for gid in ids:
            o = oracle_mod.Oracle(dict(cfg, n_games=1, game_id_base=gid), **kw)
            o.reset()
            out.append(o)
        return out

    if leg == "rollout_digest":
        env = gpu.GeneralsEnv(cfg, digest=True, actions_out=False)
        env.reset()
        for _ in range(5):
            env.rollout(32, gpu.OBS_DIGEST)
        env.torch.cuda.synchronize()
        fields = STATE_FIELDS + OUT_FIELDS + ["obs_digest"]
        got = _gather(env, fields, ids)
        for k, o in enumerate(oracles()):
            for _ in range(5):
                o.rollout(32)
            for f in fields:
                _same_game(got[f][k], np.asarray(o.field(f))[0], (leg, ids[k], f))
    elif leg == "rollout_every":
        K = 8
        env = gpu.GeneralsEnv(cfg, k_slots=K, digest=False, actions_out=False)
        env.reset()
        os_ = oracles(every_step_K=K, digest=False)
        for it in range(11):
            env.rollout(K, gpu.OBS_EVERY_STEP)
            if it not in (0, 8, 10):                       # slots compared for three of the launches, the state at the end
                for o in os_:
                    o.rollout(K, oracle_mod.OBS_EVERY_STEP)
                continue
            env.torch.cuda.synchronize()
            got = [_gather(env, OUT_FIELDS, ids, slot=k) for k in range(K)]
            for j, o in enumerate(os_):
                o.rollout(K, oracle_mod.OBS_EVERY_STEP)
                for k in range(K):
                    for f in OUT_FIELDS:
                        _same_game(got[k][f][j], np.asarray(getattr(o, f))[k][0], (leg, it, k, ids[j], f))
        got = _gather(env, STATE_FIELDS, ids)
        for j, o in enumerate(os_):
            for f in STATE_FIELDS:
                _same_game(got[f][j], np.asarray(o.field(f))[0], (leg, ids[j], f))
    elif leg == "packed":
        env = gpu.GeneralsEnv(cfg, digest=False, actions_out=False, packed=True)
        env.reset()
        T = 150
        for _ in range(T):
            env.step()
        env.torch.cuda.synchronize()
        got = _gather(env, PACKED_FIELDS, ids)
        for k, o in enumerate(oracles(digest=False)):
            for _ in range(T):
                o.step()
            for f in PACKED_FIELDS:
                _same_game(got[f][k], np.asarray(o.field(f))[0], (leg, ids[k], f))
        assert env.last_launch_register_resident
    else:                                                  # bench.py's e2e leg: pinned actions, results one step late
        T = 90
        env = gpu.GeneralsEnv(cfg, digest=False)
        env.reset()
        h_actions = torch.empty((T, N, 2), dtype=torch.int32).pin_memory()
        for t in range(T):                                 # the action stream: the device sampler's, as in bench.py
            env.step()
            h_actions[t].copy_(env.tensors["actions_out"][0], non_blocking=True)
        env.torch.cuda.synchronize()
        env.reset()
        slots = [(torch.full((N, 2), 99, dtype=torch.int8).pin_memory(), torch.full((N,), 99, dtype=torch.uint8).pin_memory())
                 for _ in range(2)]
        seen = []                                          # host results of the sampled games, every step
        for t in range(T):
            r, d = slots[t & 1]
            env.step_host_async(h_actions[t], r, d)
            if t >= 1:
                env.host_wait(1)
                pr, pd = slots[(t - 1) & 1]
                seen.append((pr.numpy()[ids].copy(), pd.numpy()[ids].copy()))
        env.host_wait(0)
        pr, pd = slots[(T - 1) & 1]
        seen.append((pr.numpy()[ids].copy(), pd.numpy()[ids].copy()))
        assert env.launch_count == 1 + T + 1 + T           # one launch per step: the kernel writes the host arrays itself
        got = _gather(env, STATE_FIELDS + OUT_FIELDS, ids)
        for k, o in enumerate(oracles(digest=False)):
            for t in range(T):
                acts = o.step(want_actions=True)
                assert np.array_equal(acts[0], h_actions[t, ids[k]].numpy()), (leg, t, ids[k], "actions")
                assert np.array_equal(seen[t][0][k], o.reward[0][0]) and seen[t][1][k] == o.done[0][0], (leg, t, ids[k])
            for f in STATE_FIELDS + OUT_FIELDS:
                _same_game(got[f][k], np.asarray(o.field(f))[0], (leg, ids[k], f))
    assert lib.gen_last_variant(env._env, None, None) == variant          # the build bench.py's leg runs
    assert int(env.tensors["episodes_done"].sum()) > 0


# ------------------------------------------------------------------------------- NEXT-1: 38-channel features (R35)
def compare_features(env, o, where=""):
    """Exact on every channel but 21 (integers and exactly rounded fp32 quotients); channel 21 = log(1 + dt) / 5
    within 1e-6 (logf is not bit-reproducible between libm and CUDA; DESIGN R35)."""
    got = env.features()
    want = o.features()
    env.torch.cuda.synchronize()
    got = got.cpu().numpy()
    assert got.shape == want.shape and got.dtype == np.float32
    for ch in range(38):
        g, w = got[:, :, ch], want[:, :, ch]
        if ch == 21:
            assert np.allclose(g, w, rtol=0, atol=1e-6), f"{where}: channel 21 off by {np.abs(g - w).max()}"
            assert np.array_equal(g == 0, w == 0), f"{where}: channel 21 zero pattern"
        elif not np.array_equal(g, w):
            bad = np.argwhere(g != w)
            raise AssertionError(f"{where}: channel {ch} differs at {bad[:5].tolist()} got {g[tuple(bad[0])]} "
                                 f"want {w[tuple(bad[0])]}")


@pytest.mark.parametrize("name,N,T,over", [
    ("c1_8x8", 64, 200, dict(auto_reset=1, max_turns=45)),                     # 8 games per CTA
    ("c1_8x8", 13, 120, dict(auto_reset=0)),                                   # frozen games, ragged last CTA
    ("c2_24x24", 37, 220, dict(max_turns=90, spawn_dmin=4)),                   # the paper-sized board
    ("c4_curriculum", 21, 160, dict(height=5, width=7, spawn_dmin=3, spawn_dmax=5, n_cities=2, max_turns=50)),
    ("c4_curriculum", 19, 160, dict(height=9, width=11, spawn_dmin=3, spawn_dmax=5, n_cities=3, max_turns=70)),
    ("c2_24x24", 5, 90, dict(height=32, width=32, max_turns=60, spawn_dmin=3)),  # largest board
    ("c2_24x24", 9, 60, dict(height=1, width=17, n_cities=1, spawn_dmin=2, max_turns=40)),   # one row
])
def test_features_match_oracle_every_turn(gpu, oracle_mod, name, N, T, over):
    """gen_features after reset and after every step against orc_features on the same play: every channel of Table
    IV, the memory across auto-resets (R17), ring wrap of the delta history, stride padding, quads that straddle
    rows (W not a multiple of 4) and ragged CTAs."""
    cfg, _ = workloads.config(name, n_games=N, **over)
    env, o = make_pair(gpu, oracle_mod, cfg)
    # the memory buffers of a fresh binding are zero; poison them to show turn 0 starts from an empty memory
    env.reset()
    o.reset()
    env.features()
    for k in ("mem_bits", "last_army", "last_seen", "hist"):
        env.feat_tensors[k].fill_(0x55 if k != "last_seen" else 7)
    env.feat_tensors["feat"].fill_(float("nan"))
    compare_features(env, o, where="reset")
    for t in range(T):
        env.step()
        o.step()
        compare_features(env, o, where=f"step {t}")
    compare(env, o, where="state untouched by gen_features")
    if cfg["auto_reset"]:
        assert int(o.episodes_done.sum()) > 0


def test_features_staged_kernel_and_errors(gpu, oracle_mod):
    """gen_features reads only the state planes and scalars, so it does not matter which kernel stepped the game
    (here the staged one: no bitboard cache), nor whether k_features was compiled for the board (here: not).
    Multi-player handles are served since R38 (test_multi_player_features_*); an empty batch launches nothing."""
    cfg, _ = workloads.config("c2_24x24", n_games=11, max_turns=64, spawn_dmin=4)
    env = gpu.GeneralsEnv(cfg, bitboards=False)
    env.set_generic(True, True)                              # the generic k_features instantiation on a 24x24 board
    o = oracle_mod.Oracle(cfg)
    env.reset()
    o.reset()
    compare_features(env, o, where="reset")
    for it in range(80):
        env.step()
        o.step()
        compare_features(env, o, where=f"it {it}")
    cfg0, _ = workloads.config("c2_24x24", n_games=0)          # an empty batch is served without a launch
    env0 = gpu.GeneralsEnv(cfg0)
    env0.reset()
    n0 = env0.launch_count
    assert env0.features().shape == (0, 2, 38, 576) and env0.launch_count == n0


def test_features_full_size_sampled_games(gpu, oracle_mod):
    """BASELINE config 2 at its full batch (16,384 games) in the launch configuration bench.py --features times:
    gen_step + gen_features every turn; the oracle replays a sample of global game ids one by one (M2)."""
    import torch
    N, T = 16384, 70
    cfg, _ = workloads.config("c2_24x24", n_games=N, max_turns=50)
    env = gpu.GeneralsEnv(cfg, digest=False, actions_out=False)
    env.reset()
    env.features()
    for _ in range(T):
        env.step()
        feat = env.features()
    env.torch.cuda.synchronize()
    ids = sorted(set(list(range(6)) + list(range(N - 6, N)) + list(range(5, N, N // 11))))
    got = feat.index_select(0, torch.tensor(ids, device=env.device)).cpu().numpy()
    for k, gid in enumerate(ids):
        o = oracle_mod.Oracle(dict(cfg, n_games=1, game_id_base=gid))
        o.reset()
        o.features()
        for _ in range(T):
            o.step()
            want = o.features()
        for ch in range(38):
            if ch == 21:
                assert np.allclose(got[k, :, ch], want[0, :, ch], rtol=0, atol=1e-6), (gid, ch)
            else:
                assert np.array_equal(got[k, :, ch], want[0, :, ch]), (gid, ch)
    # properties at any size: the four cell classes partition the board; visible army splits by owner
    HW = 576
    f = feat[:, :, :, :HW]
    assert bool(((f[:, :, 9] + f[:, :, 10] + f[:, :, 11] + f[:, :, 12]) == 1).all())
    assert bool((f[:, :, 0] == f[:, :, 1] + f[:, :, 2] + f[:, :, 3]).all())
    assert bool((f[:, :, 14] == env.tensors["turn"].float()[:, None, None]).all())


# ------------------------------------------------------------------------------- NEXT-3: official map generator (R36)
@pytest.mark.parametrize("N,T,over,staged", [
    (96, 60, dict(max_turns=25), False),                                         # the paper's parameters, frequent resets
    (96, 60, dict(max_turns=25), True),                                          # the staged kernel's generator call
    (64, 40, dict(play_min=0, spawn_dmin=3, spawn_dmax=20, spawn_exact=1, max_turns=15), False),   # curriculum in BFS steps
    (50, 30, dict(mountain_thr=workloads.thr(45), spawn_dmin=12, max_turns=10), False),  # many rejected attempts
    (40, 30, dict(height=9, width=13, play_min=5, spawn_dmin=6, n_cities=2, n_cities_max=4, castle_radius=2, max_turns=10), False),
    (40, 20, dict(height=32, width=32, play_min=20, spawn_dmin=25, n_cities=12, n_cities_max=16, max_turns=8), False),
    (30, 20, dict(height=1, width=5, play_min=0, mountain_thr=0, spawn_dmin=4, n_cities=1, n_cities_max=0, castle_radius=1, max_turns=6), False),
    (30, 20, dict(height=4, width=4, play_min=0, spawn_dmin=9, n_cities=3, n_cities_max=0, castle_radius=0, max_turns=6), False),   # infeasible window: the last attempt widens it
])
def test_official_maps_match_oracle(gpu, oracle_mod, N, T, over, staged):
    """The warp-level generator (row-word BFS) against the oracle's queue BFS: gen_reset and every auto-reset
    regeneration inside gen_step (both kernels) and inside fused rollouts produce the same boards bit for bit."""
    cfg, _ = workloads.config("official_23x23", n_games=N, **over)
    env = gpu.GeneralsEnv(cfg, bitboards=not staged)
    o = oracle_mod.Oracle(cfg)
    env.reset()
    o.reset()
    compare(env, o, where="reset")
    compare_features(env, o, where="reset")                     # Table IV's known padded border (ch 8, ch 13)
    for t in range(T):
        env.step()
        o.step()
        compare(env, o, where=f"step {t}")
        compare_features(env, o, where=f"step {t}")
    env.rollout(24, gpu.OBS_DIGEST)
    o.rollout(24, oracle_mod.OBS_DIGEST)
    compare(env, o, where="rollout")
    assert int(o.episode.min()) >= 2                           # every game was regenerated at least twice


def test_official_maps_full_size_sampled_games(gpu, oracle_mod):
    """16,384 official 23x23 maps (the batch bench.py --sweep times): sampled global ids replayed by the oracle,
    constraints of P:L79 checked on ALL maps with torch ops (castle count and garrison, two generals, padding)."""
    import torch
    N, T = 16384, 40
    cfg, _ = workloads.config("official_23x23", n_games=N, max_turns=30)
    env = gpu.GeneralsEnv(cfg, digest=False, actions_out=False)
    env.reset()
    terrain0 = env.tensors["terrain"].clone()
    army0 = env.tensors["army"].clone()
    for _ in range(T):
        env.step()
    env.torch.cuda.synchronize()
    n_castles = (terrain0 == CT).sum(1)
    assert int(n_castles.min()) >= 9 and int(n_castles.max()) <= 11
    assert bool(((terrain0 == GN).sum(1) == 2).all())
    garrison = army0[terrain0 == CT]
    assert int(garrison.min()) >= 40 and int(garrison.max()) <= 50
    dens = (terrain0[:, :529] == MT).float().mean().item()
    assert 0.2 < dens < 0.45                                    # 20 % inside the playable area plus the padding
    ids = sorted(set(list(range(8)) + list(range(N - 8, N)) + list(range(3, N, N // 17))))
    sel = torch.tensor(ids, device=env.device)
    fields = STATE_FIELDS + OUT_FIELDS
    got = {f: (env.tensors[f][0] if f in OUT_FIELDS else env.tensors[f]).index_select(0, sel).cpu().numpy() for f in fields}
    for k, gid in enumerate(ids):
        o = oracle_mod.Oracle(dict(cfg, n_games=1, game_id_base=gid))
        o.reset()
        assert np.array_equal(terrain0[gid].cpu().numpy(), o.terrain[0]), gid
        for _ in range(T):
            o.step()
        for f in fields:
            want = np.asarray(o.field(f))[0]
            have = got[f][k]
            if have.dtype != want.dtype:
                have = have.view(want.dtype)
            assert np.array_equal(have, want.reshape(have.shape)), (gid, f)


# ------------------------------------------------------------------------------- launch chaining (step_epoch)
def test_chained_launches_keep_stream_order(gpu, oracle_mod):
    """gen_step launches of one handle chain warp by warp through gen_buffers.step_epoch instead of waiting for the
    whole previous grid.  Adversarial interleaving: a large batch A and a tiny batch B stepped alternately on one
    stream (B's grid is done long before A's), with a foreign kernel (a torch copy of A's outputs) or a staged-kernel
    call on A right behind B's launch.  Every snapshot must equal the unchained run's."""
    import torch
    cfgA, _ = workloads.config("c2_24x24", n_games=16384, max_turns=40)
    cfgB, _ = workloads.config("c2_24x24", n_games=4, game_id_base=1 << 20)
    A = gpu.GeneralsEnv(cfgA, digest=False, actions_out=False)
    B = gpu.GeneralsEnv(cfgB, digest=False, actions_out=False)
    R = gpu.GeneralsEnv(cfgA, digest=False, actions_out=False)         # reference: every launch waits for the grid
    R.set_chaining(False)
    for e in (A, B, R):
        e.reset()
    names = ["obs_army", "obs_owner", "obs_vis", "army", "owner", "land", "reward", "done", "turn"]
    snaps, refs = [], []
    for t in range(60):
        A.step()
        A.step()
        B.step()
        snaps.append([A.tensors[n].clone() for n in names])             # a kernel that is not ours, behind B's launch
        R.step()
        R.step()
        torch.cuda.synchronize()
        refs.append([R.tensors[n].clone() for n in names])
        if t % 20 == 19:                                                 # a staged-kernel call on A behind B's launch
            A.step()
            B.step()
            A.rollout(3, gpu.OBS_NONE)
            A.step()
            R.step()
            R.rollout(3, gpu.OBS_NONE)
            R.step()
    torch.cuda.synchronize()
    for t, (s, r) in enumerate(zip(snaps, refs)):
        for n, a, b in zip(names, s, r):
            assert torch.equal(a, b), (t, n)
    for n in names:
        assert torch.equal(A.tensors[n], R.tensors[n]), n
    assert A.last_launch_register_resident


def test_chaining_under_graph_capture_and_replay(gpu, oracle_mod):
    """The tickets of launch chaining live on the device, so launches recorded into a CUDA graph chain as well and
    replays mix freely with eager launches: a graph of five steps replayed once between eager steps stays bit-exact
    with the oracle; further replays (same sampler counters: not a valid trajectory, but deterministic) and eager steps
    give the same tensors with chaining on and off."""
    import torch
    cfg, _ = workloads.config("c2_24x24", n_games=3000, max_turns=40, spawn_dmin=5)

    def run(chain):
        env = gpu.GeneralsEnv(cfg, digest=False)
        env.set_chaining(chain)
        env.reset()
        for _ in range(3):
            env.step()
        torch.cuda.synchronize()
        g = torch.cuda.CUDAGraph()
        side = torch.cuda.Stream()
        with torch.cuda.graph(g, stream=side):
            for _ in range(5):
                env.step()
        torch.cuda.synchronize()
        assert env.global_step == 8
        g.replay()
        for _ in range(4):
            env.step()
        torch.cuda.synchronize()
        mid = {k: v.clone() for k, v in env.tensors.items() if k != "step_epoch"}
        for _ in range(3):
            g.replay()
            g.replay()
            env.step()
            env.step()
        torch.cuda.synchronize()
        return env, mid, {k: v.clone() for k, v in env.tensors.items() if k != "step_epoch"}

    env, mid, end = run(True)
    o = oracle_mod.Oracle(cfg, digest=False)
    o.reset()
    for _ in range(12):
        o.step()
    for f in STATE_FIELDS + OUT_FIELDS:
        t = mid[f][0] if f in OUT_FIELDS else mid[f]
        got = t.cpu().numpy()
        want = np.asarray(o.field(f))
        if got.dtype != want.dtype:
            got = got.view(want.dtype)
        assert np.array_equal(got, want.reshape(got.shape)), f
    _, mid2, end2 = run(False)
    for k in end:
        assert torch.equal(end[k], end2[k]) and torch.equal(mid[k], mid2[k]), k


@pytest.mark.parametrize("name,N,T,over", [
    ("c2_24x24", 37, 150, dict(max_turns=70, spawn_dmin=4)),
    ("c1_8x8", 64, 100, dict(auto_reset=1, max_turns=45)),
    ("c4_curriculum", 21, 100, dict(height=5, width=7, spawn_dmin=3, spawn_dmax=5, n_cities=2, max_turns=50)),
])
def test_features_bf16_match_oracle(gpu, oracle_mod, name, N, T, over):
    """R37: gen_features into feat_bf16 against the oracle's fp32 tensor rounded once to bfloat16: the 16-bit patterns
    are equal on every channel but 21, which stays within one bfloat16 ulp (R35: its fp32 value is reproducible to
    1e-6 only).  Armies are inflated on the way so that values beyond bfloat16's 8 bits of mantissa occur."""
    import torch
    cfg, _ = workloads.config(name, n_games=N, **over)
    env, o = make_pair(gpu, oracle_mod, cfg)
    env.reset()
    o.reset()
    HW = cfg["height"] * cfg["width"]
    for t in range(T + 1):
        if t:
            env.step()
            o.step()
        if t % 25 == 10:                     # inflate the armies on both sides the same way, then re-derive the rest
            big = np.minimum(o.army[:, :HW].astype(np.int32) * 5 + 300, 30000).astype(np.int16)
            o.army[:, :HW] = np.where(o.owner[:, :HW] >= 0, big, o.army[:, :HW])
            o.observe()
            env.tensors["army"].copy_(torch.from_numpy(o.army))
            env.observe()
        got = env.features(bf16=True)
        want = o.features(bf16=True)
        torch.cuda.synchronize()
        assert got.dtype == torch.bfloat16
        g = got.view(torch.int16).cpu().numpy().view(np.uint16)
        for ch in range(38):
            if ch == 21:
                gf = got[:, :, ch].float().cpu().numpy()
                wf = torch.from_numpy(want[:, :, ch].view(np.int16)).view(torch.bfloat16).float().numpy()
                assert np.abs(gf - wf).max() <= 2.0 ** -7, f"turn {t}: channel 21"
            else:
                assert np.array_equal(g[:, :, ch], want[:, :, ch]), f"turn {t}: channel {ch}"
    assert (o.feat > 256).any()


def test_chaining_survives_geometry_changes(gpu, oracle_mod):
    """Tickets are per group of 4 games, not per CTA: changing the CTA size between chained launches (gen_set_launch),
    switching chaining off and on, and a batch that is not a multiple of the CTA size keep the trajectory bit-exact."""
    cfg, _ = workloads.config("c2_24x24", n_games=1021, max_turns=60, spawn_dmin=5)
    env = gpu.GeneralsEnv(cfg, digest=False)
    o = oracle_mod.Oracle(cfg, digest=False)
    env.reset()
    o.reset()
    for t in range(90):
        if t % 7 == 3:
            env.set_launch((4, 8, 16, 0)[(t // 7) % 4])
        if t % 11 == 5:
            env.set_chaining(t % 2 == 0)
        env.step()
        o.step()
        if t % 10 == 9:
            compare(env, o, digest=False, where=f"step {t}")
    compare(env, o, digest=False, where="end")


def test_features_hand_worked_example_W12_on_gpu(gpu, oracle_mod):
    """The hand-worked feature example of tests/golden/features_worked_example.txt replayed through gen_step (explicit
    actions) and gen_features: the CUDA path against the values written out by hand, not against the oracle."""
    import os
    import torch
    from helpers import hand_board
    o = hand_board(oracle_mod, 2, 3, 2, {(0, 0): (GN, 0, 5), (0, 1): (PL, 0, 3), (0, 2): (MT, -1, 0),
                                         (1, 0): (CT, -1, 42), (1, 2): (GN, 1, 7)}, turn=0)
    env = gpu.GeneralsEnv(dict(n_games=1, height=2, width=3, n_players=2, team_size=1), digest=False)
    put_board(env, o)
    moves = [None, (act(0, 1, 3, DOWN), 0), (0, act(1, 2, 3, LEFT)), (0, act(1, 1, 3, UP))]
    frames = []
    for mv in moves:
        if mv is not None:
            env.step(torch.tensor([mv], dtype=torch.int32, device=env.device))
        frames.append(env.features().cpu().numpy().copy())
    want = {}
    path = os.path.join(os.path.dirname(__file__), "golden", "features_worked_example.txt")
    for line in open(path):
        if line.startswith("#") or not line.strip():
            continue
        tok = line.split()
        want.setdefault((int(tok[0]), int(tok[1])), {})[int(tok[2])] = np.array([float(x) for x in tok[3:]], np.float32)
    for (fr, p), chans in want.items():
        for ch in range(38):
            got = frames[fr][0, p, ch, :6]
            exp = chans.get(ch, np.zeros(6, np.float32))
            if ch == 21:
                assert np.allclose(got, exp, atol=1e-6), (fr, p, ch, got)
            else:
                assert np.array_equal(got, exp), (fr, p, ch, got, exp)
        assert not frames[fr][0, p, :, 6:].any()


@pytest.mark.parametrize("name,N,T,over,bf16", [
    ("c5a_2v2", 9, 120, dict(max_turns=60), False),                                   # 2v2 on 32x32: team visibility
    ("c5b_ffa8", 5, 100, dict(max_turns=60), False),                                  # 8 players: 2,048 items per game
    ("c5b_ffa8", 7, 120, dict(n_players=3, height=7, width=9, n_cities=2, spawn_dmin=3, max_turns=40), False),
    ("c5a_2v2", 6, 80, dict(height=12, width=13, n_cities=3, spawn_dmin=3, max_turns=40), True),
])
def test_multi_player_features_match_oracle(gpu, oracle_mod, name, N, T, over, bf16):
    """R38: the feature tensor with more than two players (k_features_mp) against the oracle, every channel every
    turn: team visibility, any enemy as "the opponent", enemy sums on the scoreboard channels."""
    import torch
    cfg, _ = workloads.config(name, n_games=N, **over)
    env, o = make_pair(gpu, oracle_mod, cfg)
    env.reset()
    o.reset()
    for t in range(T + 1):
        if t:
            env.step()
            o.step()
        if not bf16:
            compare_features(env, o, where=f"turn {t}")
            continue
        got = env.features(bf16=True)
        want = o.features(bf16=True)
        torch.cuda.synchronize()
        gb = got.view(torch.int16).cpu().numpy().view(np.uint16)
        for ch in range(38):
            if ch == 21:
                gf = got[:, :, ch].float().cpu().numpy()
                wf = torch.from_numpy(want[:, :, ch].view(np.int16)).view(torch.bfloat16).float().numpy()
                assert np.abs(gf - wf).max() <= 2.0 ** -7
            else:
                assert np.array_equal(gb[:, :, ch], want[:, :, ch]), (t, ch)
    assert int(o.episodes_done.sum()) > 0


@pytest.mark.parametrize("name,over", [("c4_curriculum", dict()), ("official_23x23", dict(play_min=0))])
def test_spawn_curriculum_raised_over_time(gpu, oracle_mod, name, over):
    """the cap on the spawn distance starts small and is raised over training.  gen_set_spawn changes the window
    of the boards generated from then on (auto-resets included) on the same handle; the oracle follows by changing the
    same three config fields; boards stay bit-exact and the generals' distance tracks the window."""
    cfg, _ = workloads.config(name, n_games=48, max_turns=12, spawn_dmin=3, spawn_dmax=4, spawn_exact=0, **over)
    env, o = make_pair(gpu, oracle_mod, cfg)
    env.reset()
    o.reset()
    W = cfg["width"]
    for stage, (lo, hi) in enumerate([(3, 4), (3, 8), (6, 14), (17, 0)]):
        env.set_spawn(lo, hi, 0)
        o.cfg.spawn_dmin, o.cfg.spawn_dmax, o.cfg.spawn_exact = lo, hi, 0
        for t in range(13):                                      # every game is truncated and regenerated once
            env.step()
            o.step()
        compare(env, o, where=f"stage {stage}")
        gc = o.general_cell.astype(int)
        d = np.abs(gc[:, 0] // W - gc[:, 1] // W) + np.abs(gc[:, 0] % W - gc[:, 1] % W)
        assert (o.turn <= 4).all()                               # every board on the table was drawn in this stage
        if name == "c4_curriculum":                              # Manhattan window (R29)
            assert d.min() >= lo and (hi == 0 or d.max() <= hi)
        else:                                                    # BFS steps >= Manhattan distance (R36)
            assert hi == 0 or d.max() <= hi
    with pytest.raises(gpu.GenError):
        env.set_spawn(5, 3, 0)


def test_random_configurations_fuzz(gpu, oracle_mod):
    """Seeded differential fuzz: 90 random configurations (board 2..32 x 2..32, 2..8 players, team sizes, rule flags,
    both generators, policies, truncation, packed observation, history ring, kernel choice), each stepped for 40 turns
    with an explicit-action turn and a fused rollout mixed in, every tensor compared with the oracle every few turns,
    the feature tensor on the way."""
    import torch
    rng = np.random.default_rng(20260623)
    done_eps = 0
    for case in range(90):
        P = int(rng.choice([2, 2, 2, 3, 4, 4, 6, 8]))
        H, W = int(rng.integers(2, 33)), int(rng.integers(2, 33))
        if H * W < 4 * P:
            H, W = max(H, 6), max(W, 6)
        team_size = int(rng.choice([t for t in (1, 2, 4) if t <= P and (t == 1 or P % t == 0) and P // t >= 2] or [1]))
        official = P == 2 and rng.random() < 0.35 and H >= 4 and W >= 4
        cfg = dict(n_games=int(rng.integers(1, 40)), height=H, width=W, n_players=P, team_size=team_size,
                   n_cities=int(rng.integers(0, max(1, H * W // 12) + 1)), city_army_lo=int(rng.integers(0, 30)),
                   city_army_hi=int(rng.integers(30, 60)), spawn_dmin=int(rng.integers(0, max(1, (H + W) // 3) + 1)),
                   spawn_dmax=0, spawn_exact=0, max_turns=int(rng.choice([0, 7, 20])), auto_reset=int(rng.integers(0, 2)),
                   rule_flags=int(rng.integers(0, 8)), game_id_base=int(rng.integers(0, 1 << 30)),
                   mountain_thr=workloads.thr(int(rng.integers(0, 45))), seed=int(rng.integers(0, 1 << 62)),
                   pass_thr=workloads.thr(int(rng.integers(0, 30))), half_thr=workloads.thr(int(rng.integers(0, 101))),
                   bias_thr=workloads.thr(int(rng.choice([0, 0, 50, 100]))))
        if official:
            cfg.update(map_mode=1, n_cities_max=cfg["n_cities"] + int(rng.integers(0, 3)),
                       play_min=int(rng.choice([0, min(H, W, 3), min(H, W)])), castle_radius=int(rng.integers(0, 7)))
        packed, history = bool(rng.random() < 0.3), bool(rng.random() < 0.3)
        staged = bool(rng.random() < 0.3)
        env = gpu.GeneralsEnv(cfg, packed=packed, history=history, bitboards=not staged, digest=bool(rng.random() < 0.5))
        o = oracle_mod.Oracle(cfg, digest="obs_digest" in env.tensors)
        env.reset()
        o.reset()
        fields = ([f for f in ALL_FIELDS if f in env.tensors] + (["obs_packed"] if packed else [])
                  + (["score_hist"] if history else []))
        where = f"case {case}: {cfg}"
        dg = "obs_digest" in env.tensors
        compare(env, o, fields=fields, digest=dg, where=where + " reset")
        feats = case % 3 == 0                                     # the feature tensor every turn (R35, R38)
        if feats:
            compare_features(env, o, where=where + " reset")
        for t in range(40):
            if t == 13:
                a = workloads.random_actions(rng, cfg["n_games"], P, H, W)
                env.step(torch.from_numpy(a).to(env.device))
                o.step(a)
            elif t == 27 and not feats:                               # (one gen_features call per turn: no rollouts then)
                env.rollout(3, gpu.OBS_DIGEST if dg else gpu.OBS_NONE)
                o.rollout(3, oracle_mod.OBS_DIGEST if dg else oracle_mod.OBS_NONE)
                if not dg:                                        # a state-only rollout leaves no observation
                    env.step()
                    o.step()
            else:
                env.step()
                o.step()
            if feats:
                compare_features(env, o, where=where + f" t={t}")
            if t % 9 == 8 or t == 39:
                compare(env, o, fields=fields, digest=dg, where=where + f" t={t}")
        done_eps += int(o.episodes_done.sum())
    assert done_eps > 0


# ------------------------------------------------------------------------------- temporal tokens (R39)
@pytest.mark.parametrize("name,N,T,over", [
    ("c2_24x24", 45, 620, dict(max_turns=0, auto_reset=0)),                    # one long episode: the ring wraps
    ("c4_curriculum", 37, 300, dict(height=10, width=10, spawn_dmin=3, spawn_dmax=5, n_cities=3, max_turns=90)),
    ("c5a_2v2", 9, 120, dict(height=12, width=12, n_cities=3, spawn_dmin=4, max_turns=50)),
    ("c5b_ffa8", 5, 90, dict(height=12, width=13, n_players=3, spawn_dmin=4, n_cities=4, max_turns=40)),
])
def test_history_windows_match_oracle(gpu, oracle_mod, name, N, T, over):
    """gen_history_windows (the two 512-step windows behind the temporal tokens) against orc_history_windows
    on the same play: oldest first, zeros before the episode's first turn, leftovers of earlier episodes masked,
    enemies summed for more than two players (R38), before and after the ring wraps; the output buffer is poisoned
    before every call."""
    cfg, _ = workloads.config(name, n_games=N, **over)
    env = gpu.GeneralsEnv(cfg, digest=False, history=True)
    o = oracle_mod.Oracle(cfg)
    env.reset()
    o.reset()
    out = env.torch.full((N, cfg["n_players"], 2, 512), -77, dtype=env.torch.int32, device=env.device)
    for t in range(T):
        env.step()
        o.step()
        if t % 37 == 0 or t >= T - 3 or t in (509, 510, 511, 512, 513):
            out.fill_(-77)
            got = env.history_windows(out).cpu().numpy()
            assert np.array_equal(got, o.history_windows()), f"{name}: windows differ at step {t}"
    if cfg["max_turns"]:
        assert int(o.episodes_done.sum()) > 0
    no_ring = gpu.GeneralsEnv(cfg, digest=False)                # without the ring the call is refused
    with pytest.raises(gpu.GenError):
        no_ring.history_windows()


def test_history_windows_empty_batch(gpu):
    cfg, _ = workloads.config("c2_24x24", n_games=0)
    env = gpu.GeneralsEnv(cfg, history=True)
    assert env.history_windows().shape == (0, 2, 2, 512)


# ------------------------------------------------------------------------------- sanitizer target
def test_sanitizer_coverage_run(gpu, oracle_mod):
    """One short run over every kernel of the library, small enough for compute-sanitizer:
        compute-sanitizer --tool {memcheck,racecheck,synccheck,initcheck} \\
            python -m pytest tests/test_gpu_parity.py -q -k sanitizer_coverage_run
    (summaries under profiles/).  Config 1 (8x8) and a 24x24 batch with a ragged last CTA: gen_reset, chained
    gen_step launches (k_step: tickets, TMA row loads, 32-bit reductions on int16 pairs), gen_step with explicit
    actions, gen_rollout(8) with the digest, gen_observe, gen_sample, reset and auto-reset with the official
    generator, gen_features in both instantiations (fp32 1v1, bfloat16; the multi-player kernel).  It is a parity
    test in its own right: everything is compared with the oracle."""
    import torch
    for name, N, over in (("c1_8x8", 21, dict(auto_reset=1, max_turns=12)),
                          ("c2_24x24", 21, dict(max_turns=14)),
                          ("official_23x23", 13, dict(max_turns=9))):
        cfg, _ = workloads.config(name, n_games=N, **over)
        env = gpu.GeneralsEnv(cfg, digest=False)
        o = oracle_mod.Oracle(cfg)
        env.reset()
        o.reset()
        compare_features(env, o, where=f"{name} reset")
        for t in range(3):                                     # three chained launches, nothing in between
            env.step()
            o.step()
        compare(env, o, digest=False, where=f"{name} chained steps")
        for t in range(16):
            env.step()
            o.step()
            compare_features(env, o, where=f"{name} step {t}")
        a = o.sample()
        assert np.array_equal(env.sample().cpu().numpy(), a)
        env.step(torch.from_numpy(a).to(env.device))
        o.step(a)
        env.observe()
        compare(env, o, digest=False, where=f"{name} explicit actions + observe")
        assert env.last_launch_register_resident is False      # gen_observe is the staged kernel
        env.close()
    cfg, _ = workloads.config("c2_24x24", n_games=19, max_turns=11)
    env, o = make_pair(gpu, oracle_mod, cfg)
    env.reset()
    o.reset()
    env.rollout(8, gpu.OBS_DIGEST)
    o.rollout(8, oracle_mod.OBS_DIGEST)
    env.step()
    o.step()
    compare(env, o, where="rollout(8) + staged step with digest")
    bf = env.features(bf16=True)
    torch.cuda.synchronize()
    assert bf.dtype == torch.bfloat16 and bool(torch.isfinite(bf.float()).all())
    cfg, _ = workloads.config("c5a_2v2", n_games=6, height=12, width=12, n_cities=3, spawn_dmin=4, max_turns=10)
    env, o = make_pair(gpu, oracle_mod, cfg)
    env.reset()
    o.reset()
    for t in range(12):
        env.step()
        o.step()
        compare_features(env, o, where=f"2v2 step {t}")
    compare(env, o, where="2v2")


# ------------------------------------------------------------------------------- memory discipline without a sanitizer
def test_guard_bands_and_poisoned_outputs(gpu, oracle_mod):
    """compute-sanitizer is closed on this GPU pool (profiles/r02_sanitizer.md), so the checks it would make are made
    by hand.  (1) memcheck's part: every device buffer of the handle is carved out of a larger allocation filled with
    0xA5 -- 4 KB of guard band on both sides, also around the feature buffers and the window output -- and the bands
    must be untouched after resets, chained steps, explicit-action steps, fused rollouts, gen_observe, gen_sample,
    gen_features and gen_history_windows on every kernel variant a ragged batch reaches.  (2) initcheck's part:
    every OUTPUT buffer is poisoned before each call, so a cell the kernels fail to write shows up as a mismatch
    with the oracle.  Boards: 24x24 1v1 (board-specialised kernels), 23x23 official maps, 12x13 with 3 players
    (generic kernels, stride padding), 32x32 2v2."""
    import ctypes as C
    import torch
    GUARD = 4096
    OUT = ["reward", "done", "winner", "obs_army", "obs_owner", "obs_terrain", "obs_vis", "actions_out"]

    def fence(env):
        """Move every tensor of env into the middle of a poisoned allocation; returns the guard checkers."""
        bands = []
        for name, t in list(env.tensors.items()):
            nbytes = t.numel() * t.element_size()
            raw = torch.full((nbytes + 2 * GUARD,), 0xA5, dtype=torch.uint8, device=env.device)
            mid = raw[GUARD:GUARD + nbytes]
            mid.copy_(t.view(torch.uint8).reshape(-1))
            view = mid.view(t.dtype).reshape(t.shape)
            assert view.data_ptr() % 16 == 0
            env.tensors[name] = view
            setattr(env, name, view)
            setattr(env.bufs, name, view.data_ptr())
            bands.append((name, raw, nbytes))
        return bands

    def check(bands, where):
        torch.cuda.synchronize()
        for name, raw, nbytes in bands:
            assert bool((raw[:GUARD] == 0xA5).all()) and bool((raw[GUARD + nbytes:] == 0xA5).all()), \
                f"{where}: write outside {name}"

    def poison(env):
        for name in OUT:
            if name in env.tensors:
                env.tensors[name].view(torch.uint8).fill_(0x5A)

    cases = [("c2_24x24", 37, dict(max_turns=25), True), ("official_23x23", 21, dict(max_turns=20), True),
             ("c5b_ffa8", 11, dict(height=12, width=13, n_players=3, spawn_dmin=4, n_cities=4, max_turns=30), True),
             ("c5a_2v2", 7, dict(max_turns=20), False)]
    for name, N, over, digest in cases:
        cfg, _ = workloads.config(name, n_games=N, **over)
        for step_kernel in (True, False):
            use_digest = digest and not step_kernel
            env = gpu.GeneralsEnv(cfg, digest=use_digest, history=True, bitboards=step_kernel)
            if step_kernel:
                env.set_generic(False, -1)
            o = oracle_mod.Oracle(cfg)
            bands = fence(env)
            poison(env)
            env.reset()
            o.reset()
            compare(env, o, digest=False, where=f"{name} reset")
            for t in range(30):
                poison(env)
                if t % 5 == 4:
                    a = o.sample()
                    env.step(torch.from_numpy(a).to(env.device))
                    o.step(a)
                else:
                    env.step()
                    o.step()
                compare(env, o, digest=False, where=f"{name} step {t}")
            assert env.last_launch_register_resident == step_kernel
            poison(env)
            env.rollout(7, gpu.OBS_DIGEST if use_digest else gpu.OBS_NONE)
            o.rollout(7, oracle_mod.OBS_DIGEST if use_digest else oracle_mod.OBS_NONE)
            assert np.array_equal(env.sample().cpu().numpy(), o.sample())
            poison(env)
            env.observe()
            compare(env, o, fields=STATE_FIELDS + OUT_FIELDS[3:], digest=False, where=f"{name} rollout + observe")
            # feature tensor and windows, their buffers fenced too
            env.features()
            fb = []
            for k, t in list(env.feat_tensors.items()):
                nbytes = t.numel() * t.element_size()
                raw = torch.full((nbytes + 2 * GUARD,), 0xA5, dtype=torch.uint8, device=env.device)
                mid = raw[GUARD:GUARD + nbytes]
                mid.copy_(t.view(torch.uint8).reshape(-1))
                view = mid.view(t.dtype).reshape(t.shape)
                env.feat_tensors[k] = view
                setattr(env.feat_bufs, k, view.data_ptr())
                fb.append((k, raw, nbytes))
            env.feat = env.feat_tensors["feat"]
            env.feat.fill_(float("nan"))
            f = env.features()
            torch.cuda.synchronize()
            assert bool(torch.isfinite(f).all())
            wraw = torch.full((N * cfg["n_players"] * 2 * 512 * 4 + 2 * GUARD,), 0xA5, dtype=torch.uint8, device=env.device)
            win = wraw[GUARD:-GUARD].view(torch.int32).reshape(N, cfg["n_players"], 2, 512)
            assert np.array_equal(env.history_windows(win).cpu().numpy(), o.history_windows())
            check(bands + fb + [("windows", wraw, wraw.numel() - 2 * GUARD)], f"{name} step_kernel={step_kernel}")
            env.close()
