"""Host-only checks of the C-ABI library: it loads, exports every symbol include/generals.h declares,
validates configurations and reports sizes.  No kernel is launched (no GPU needed)."""
import ctypes as C
import os
import re

import pytest

import workloads
from paper_2606_23348_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.load_library()


def test_exports_every_declared_symbol(lib):
    header = open(os.path.join(ROOT, "include", "generals.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b(gen_[a-z_]+)\s*\(", header))
    assert declared == set(binding.EXPORTS)
    for name in declared:
        assert hasattr(lib, name), name
    assert b"sm_100a" in lib.gen_version()


def binding_err(name):
    return {"GEN_ERR_NULL": -1, "GEN_ERR_CONFIG": -2, "GEN_ERR_ALIGN": -3, "GEN_ERR_ARG": -4, "GEN_ERR_CUDA": -5,
            "GEN_ERR_SIZE": -6}[name]


def test_struct_layouts_match_header():
    assert C.sizeof(binding.GenConfig) == 13 * 4 + 3 * 4 + 8 + 4 * 4
    assert C.sizeof(binding.GenBuffers) == 29 * 8
    assert C.sizeof(binding.GenSizes) == 8 + 29 * C.sizeof(C.c_size_t) + 8      # + bitboard_row_words, padding
    assert C.sizeof(binding.GenFeatBuffers) == 6 * 8
    assert C.sizeof(binding.GenFeatSizes) == 8 + 7 * C.sizeof(C.c_size_t)


def test_query_feat_sizes(lib):
    cfg, _ = binding.make_config(workloads.config("c2_24x24")[0])
    s = binding.GenFeatSizes()
    assert lib.gen_query_feat_sizes(C.byref(cfg), C.byref(s)) == 0
    N, S = 16384, 576
    assert s.channels == 38 and s.plane_stride == S
    assert s.feat == N * 2 * 38 * S * 4 and s.mem_bits == N * 2 * S and s.last_army == N * 2 * S * 2
    assert s.last_seen == N * 2 * S * 4 and s.hist == N * 2 * 8 * 2 * S * 2 and s.feat_bf16 == N * 2 * 38 * S * 2
    assert s.hist_windows == N * 2 * 2 * 512 * 4
    cfg4, _ = binding.make_config(workloads.config("c5a_2v2")[0])          # R38: P players, 32x32
    assert lib.gen_query_feat_sizes(C.byref(cfg4), C.byref(s)) == 0
    assert s.feat == 32768 * 4 * 38 * 1024 * 4 and s.hist == 32768 * 4 * 8 * 2 * 1024 * 2
    assert lib.gen_query_feat_sizes(None, C.byref(s)) == binding_err("GEN_ERR_NULL")


def test_query_sizes(lib):
    cfg, _ = binding.make_config(workloads.config("c2_24x24")[0])
    s = binding.GenSizes()
    assert lib.gen_query_sizes(C.byref(cfg), 1, C.byref(s)) == 0
    N, P, S = 16384, 2, 576
    assert s.plane_stride == S and s.alignment == 16
    assert s.army == N * S * 2 and s.owner == N * S and s.terrain == N * S
    assert s.obs_army == N * P * S * 2 and s.obs_vis == N * P * S
    assert s.reward == N * P and s.done == N and s.obs_digest == 8 * N
    assert s.bitboard_row_words == 24 and s.bitboards == N * (P + 3) * 24 * 4       # ceil(576 / 32) = 18 -> 24
    assert lib.gen_query_sizes(C.byref(cfg), 32, C.byref(s)) == 0
    assert s.obs_owner == 32 * N * P * S and s.army == N * S * 2
    cfg5, _ = binding.make_config(workloads.config("c1_8x8", height=5, width=7)[0])
    assert lib.gen_query_sizes(C.byref(cfg5), 1, C.byref(s)) == 0
    assert s.plane_stride == 48          # round_up(35, 16)


@pytest.mark.parametrize("bad", [dict(height=0), dict(height=33), dict(width=40), dict(n_players=1),
                                 dict(n_players=9), dict(team_size=0), dict(team_size=3),
                                 dict(city_army_lo=60), dict(n_cities=-1), dict(spawn_exact=1, spawn_dmax=0),
                                 dict(spawn_dmax=2), dict(rule_flags=64), dict(max_turns=-5),
                                 dict(n_games=-1), dict(city_army_hi=40000), dict(map_mode=2), dict(play_min=3),
                                 dict(map_mode=1, n_players=4), dict(map_mode=1, n_cities=10, n_cities_max=9),
                                 dict(map_mode=1, height=1, width=8, play_min=1)])
def test_bad_config_is_rejected(lib, bad):
    cfg, _ = binding.make_config(workloads.config("c1_8x8", **bad)[0])
    env = C.c_void_p()
    assert lib.gen_init(C.byref(cfg), C.byref(env)) == -2            # GEN_ERR_CONFIG
    assert not env.value
    s = binding.GenSizes()
    assert lib.gen_query_sizes(C.byref(cfg), 1, C.byref(s)) == -2


def test_init_argument_errors_without_gpu(lib):
    cfg, _ = binding.make_config(workloads.config("c1_8x8")[0])
    env = C.c_void_p()
    assert lib.gen_init(None, C.byref(env)) == -1
    assert lib.gen_init(C.byref(cfg), C.byref(env)) == 0 and env.value
    bufs = binding.GenBuffers()                                       # all NULL
    assert lib.gen_step(env, C.byref(bufs), None, None) == -1         # GEN_ERR_NULL, nothing launched
    assert lib.gen_reset(env, C.byref(bufs), 0, None) == -1
    assert lib.gen_reset(env, C.byref(bufs), 8, None) == -4           # unknown flag
    assert lib.gen_rollout(env, C.byref(bufs), 0, 0, None) == -4      # K <= 0
    assert lib.gen_rollout(env, C.byref(bufs), 4, 7, None) == -4      # unknown obs mode
    for name, _, _ in binding.BUFFERS:
        setattr(bufs, name, 0x1000)
    bufs.owner = 0x1008                                               # misaligned
    assert lib.gen_step(env, C.byref(bufs), None, None) == -3         # GEN_ERR_ALIGN
    assert lib.gen_set_launch(env, 3) == -4 and lib.gen_set_launch(env, 4) == 0
    assert lib.gen_launch_count(env) == 0
    assert lib.gen_set_global_step(env, 41) == 0 and lib.gen_global_step(env) == 41
    assert lib.gen_set_spawn(env, 3, 6, 0) == 0 and lib.gen_set_spawn(env, 6, 3, 0) == -2   # dmax < dmin
    assert lib.gen_set_spawn(env, 3, 0, 1) == -2 and lib.gen_set_spawn(None, 3, 0, 0) == -1  # exact needs dmax
    assert lib.gen_set_chaining(env, 0) == 0 and lib.gen_set_chaining(None, 1) == -1
    fb = binding.GenFeatBuffers()                                     # all NULL
    assert lib.gen_features(env, C.byref(bufs), C.byref(fb), None) == -3   # owner is still misaligned
    bufs.owner = 0x1000
    assert lib.gen_features(env, C.byref(bufs), C.byref(fb), None) == -1
    assert lib.gen_features(env, C.byref(bufs), None, None) == -1
    assert lib.gen_history_windows(env, C.byref(bufs), None, None) == -1          # no output buffer
    assert lib.gen_history_windows(env, C.byref(bufs), 0x1008, None) == -3        # misaligned output
    bufs.score_hist = None
    assert lib.gen_history_windows(env, C.byref(bufs), 0x1000, None) == -1        # the ring is required
    for code in (0, -1, -2, -3, -4, -5, -6, -99):
        assert lib.gen_error_string(code)
    lib.gen_destroy(env)


def test_step_noalloc_argument_errors_without_gpu(lib):
    """gen_step_noalloc refuses what it cannot serve before it touches the device: missing pointers, a batch beyond
    its built-in 8 MiB scratch array (GEN_ERR_SIZE), a digest buffer or more than four players (GEN_ERR_ARG)."""
    assert binding.NOALLOC_SCRATCH_BYTES == 8 << 20
    header = open(os.path.join(ROOT, "include", "generals.h")).read()
    assert "#define GEN_NOALLOC_SCRATCH_BYTES (8u << 20)" in header and "GEN_ERR_SIZE = -6" in header
    bufs = binding.GenBuffers()                                       # all NULL
    for over, want in ((dict(n_games=17476), "GEN_ERR_NULL"),         # fits; the planes are missing
                       (dict(n_games=17477), "GEN_ERR_SIZE"),
                       (dict(n_games=1 << 20), "GEN_ERR_SIZE")):
        cfg, _ = binding.make_config(workloads.config("c2_24x24", **over)[0])
        env = C.c_void_p()
        assert lib.gen_init(C.byref(cfg), C.byref(env)) == 0
        assert lib.gen_step_noalloc(env, C.byref(bufs), None, None) == binding_err(want)
        assert lib.gen_step_noalloc(env, None, None, None) == binding_err("GEN_ERR_NULL")
        assert lib.gen_global_step(env) == 0 and lib.gen_launch_count(env) == 0
        lib.gen_destroy(env)
    assert lib.gen_step_noalloc(None, C.byref(bufs), None, None) == binding_err("GEN_ERR_NULL")
    cfg, _ = binding.make_config(workloads.config("c5b_ffa8", n_games=8)[0])
    env = C.c_void_p()
    assert lib.gen_init(C.byref(cfg), C.byref(env)) == 0
    assert lib.gen_step_noalloc(env, C.byref(bufs), None, None) == binding_err("GEN_ERR_ARG")     # 8 players
    lib.gen_destroy(env)
    cfg, _ = binding.make_config(workloads.config("c1_8x8")[0])
    assert lib.gen_init(C.byref(cfg), C.byref(env)) == 0
    bufs.obs_digest = 0x1000
    assert lib.gen_step_noalloc(env, C.byref(bufs), None, None) == binding_err("GEN_ERR_ARG")     # digest buffer
    bufs.obs_digest = None
    bufs.army, bufs.owner, bufs.terrain = 0x1000, 0x1008, 0x1000
    assert lib.gen_step_noalloc(env, C.byref(bufs), None, None) == binding_err("GEN_ERR_ALIGN")
    assert b"GEN_NOALLOC_SCRATCH_BYTES" in lib.gen_error_string(-6)
    lib.gen_destroy(env)


def test_missing_library_fails_loudly(tmp_path):
    with pytest.raises(binding.GenError):
        binding.load_library(str(tmp_path / "nope.so"))
