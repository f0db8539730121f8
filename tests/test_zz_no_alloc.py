"""gen_step_noalloc: the step for callers that cannot allocate device memory.

Some users of this library are not in a position to call cudaMalloc when they step their games: an environment
wrapped as an operator inside another system's executor gets operands and results and no workspace; a process whose
learner took all of HBM at start-up has nothing left to allocate; an actor loop cannot afford the device-wide
synchronisation that cudaMalloc / cudaFree bring.  For them the library keeps the per-step kernel's working memory
(the bitboard cache) in a fixed 8 MiB device array of its own, shared by every call in the process.

What is checked here: the entry point gives exactly what gen_step gives with a caller-allocated cache -- every state
plane, observation plane, scoreboard, reward and done flag, bit for bit (integer work: the tolerance of this suite is
equality) -- on two calls in a row and beyond, also when another handle with a different board has used the shared
array in between (its leftovers must never be read), and that a batch beyond the array's size is refused.

The file sorts last on purpose (pytest -x stops at the first failure), and it passes alone in a fresh process as well
as after the rest of the suite: every call rebuilds what it reads, nothing depends on the array's earlier contents.
"""
import ctypes as C

import numpy as np
import pytest

from helpers import OUT_FIELDS, STATE_FIELDS
import workloads

pytestmark = pytest.mark.gpu

FIELDS = STATE_FIELDS + OUT_FIELDS + ["actions_out"]


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device")
    import paper_2606_23348_b200 as g
    g.load_library()
    return g


def same(a, b, where):
    a.torch.cuda.synchronize()
    for f in FIELDS:
        x, y = a.field(f), b.field(f)
        assert np.array_equal(x, y), f"{where}: {f} differs at {np.argwhere(x != y)[:4].tolist()}"


def pair(gpu, cfg):
    """The existing path (caller-allocated cache, its launches chained) and the no-allocation path: the second
    environment owns no cache, no chaining counters and no stack cache at all."""
    ref = gpu.GeneralsEnv(cfg, digest=False)
    na = gpu.GeneralsEnv(cfg, digest=False, bitboards=False, chain=False, stack_cache=False)
    assert "bitboards" not in na.tensors and "step_epoch" not in na.tensors and "stack_cache" not in na.tensors
    ref.reset()
    na.reset()
    same(ref, na, "reset")
    return ref, na


@pytest.mark.parametrize("name,over", [
    ("c2_24x24", dict(n_games=333, max_turns=30)),                      # the headline board, a ragged batch
    ("c1_8x8", dict(n_games=64)),
    ("c4_curriculum", dict(n_games=150, max_turns=25)),                 # biased sampler without the stack cache
    ("c5a_2v2", dict(n_games=37, max_turns=20)),                        # four players, 32x32
    ("c1_8x8", dict(n_games=50, height=5, width=7, spawn_dmin=3)),      # plane stride 48 > 35 cells
    ("official_23x23", dict(n_games=90, max_turns=20)),                 # cells past the board inside the last word
])
def test_two_calls_in_a_row_equal_gen_step(gpu, name, over):
    cfg, _ = workloads.config(name, **over)
    ref, na = pair(gpu, cfg)
    for call in range(2):                                   # the two calls in a row
        ref.step()
        na.step_noalloc()
        same(ref, na, f"{name}: call {call}")
    assert na.last_launch_register_resident                 # the scratch-backed kernel ran, not the staged one
    assert na.launch_count == 1 + 2 * 2                     # reset + (rows + step) per call
    for t in range(2, 40):                                  # ... through truncations and auto-resets
        ref.step()
        na.step_noalloc()
    same(ref, na, f"{name}: 40 calls")
    assert na.global_step == ref.global_step == 40


def test_explicit_actions_and_a_foreign_user_of_the_array(gpu):
    """Another handle (other board, other batch) steps through the same array between our calls."""
    import torch
    cfg, _ = workloads.config("c2_24x24", n_games=203, max_turns=0)
    ref, na = pair(gpu, cfg)
    other_cfg, _ = workloads.config("c5a_2v2", n_games=64, max_turns=0)
    other_ref, other = pair(gpu, other_cfg)
    rng = np.random.default_rng(11)
    for t in range(30):
        if t % 2:
            a = torch.from_numpy(workloads.random_actions(rng, 203, 2, 24, 24)).to(ref.device)
            ref.step(a)
            other.step_noalloc()
            na.step_noalloc(a)
        else:
            ref.step()
            other.step_noalloc()
            na.step_noalloc()
        other_ref.step()
        same(ref, na, f"turn {t}")
    same(other_ref, other, "the other handle")


def test_size_limit_is_enforced(gpu):
    """8 MiB holds 17,476 games of 24x24 1v1 (480 bytes each): config 2 fits, one game more than the limit does not,
    and the refusal comes before anything is launched or changed."""
    lib = gpu.load_library()
    per_game = 5 * 24 * 4
    n_max = gpu.binding.NOALLOC_SCRATCH_BYTES // per_game
    assert n_max == 17476
    cfg, _ = workloads.config("c2_24x24", n_games=n_max + 1, max_turns=0)
    env = gpu.GeneralsEnv(cfg, digest=False, bitboards=False, chain=False, stack_cache=False)
    env.reset()
    env.torch.cuda.synchronize()
    before = env.field("turn").copy()
    launches = env.launch_count
    code = lib.gen_step_noalloc(env._env, C.byref(env.bufs), None, None)
    assert code == gpu.binding.GEN_ERR_SIZE and b"GEN_NOALLOC_SCRATCH_BYTES" in lib.gen_error_string(code)
    with pytest.raises(gpu.GenError):
        env.step_noalloc()
    env.torch.cuda.synchronize()
    assert env.launch_count == launches and env.global_step == 0 and np.array_equal(env.field("turn"), before)
    env.close()
    cfg, _ = workloads.config("c2_24x24", n_games=n_max, max_turns=0)      # exactly the limit
    ref, na = pair(gpu, cfg)
    for call in range(2):
        ref.step()
        na.step_noalloc()
    same(ref, na, "at the limit")
    digest_env = gpu.GeneralsEnv(workloads.config("c1_8x8")[0], bitboards=False)     # has a digest buffer
    assert lib.gen_step_noalloc(digest_env._env, C.byref(digest_env.bufs), None, None) == -4
    ffa, _ = workloads.config("c5b_ffa8", n_games=8)
    ffa_env = gpu.GeneralsEnv(ffa, digest=False, bitboards=False)                    # more than four players
    assert lib.gen_step_noalloc(ffa_env._env, C.byref(ffa_env.bufs), None, None) == -4
