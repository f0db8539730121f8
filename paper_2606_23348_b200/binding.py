"""ctypes binding of include/generals.h.  Argument marshalling only.

The product path fails loudly when the CUDA library is missing: there is no CPU fallback and this
module never imports anything from oracle/.
"""
import ctypes as C
import os

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libgenerals.so")

OBS_DIGEST, OBS_EVERY_STEP, OBS_NONE = 0, 1, 2
GEN_KEEP_EPISODE = 1
RULE_TICK_PLAIN_ONLY, RULE_CAPTURE_HALF_FLOOR, RULE_ROTATE_PRIORITY = 1, 2, 4
GEN_ERR_SIZE = -6
NOALLOC_SCRATCH_BYTES = 8 << 20     # GEN_NOALLOC_SCRATCH_BYTES: the array behind gen_step_noalloc

EXPORTS = ["gen_query_sizes", "gen_init", "gen_set_policy", "gen_set_spawn", "gen_global_step", "gen_set_global_step",
           "gen_reset", "gen_step", "gen_step_noalloc", "gen_rollout", "gen_observe", "gen_sample", "gen_step_host",
           "gen_step_host_async", "gen_host_wait", "gen_forget_host_buffers",
           "gen_query_feat_sizes", "gen_features", "gen_history_windows",
           "gen_set_launch", "gen_set_generic", "gen_set_chaining", "gen_last_variant",
           "gen_launch_count", "gen_last_cuda_error", "gen_destroy",
           "gen_error_string", "gen_version"]


class GenError(RuntimeError):
    pass


class GenConfig(C.Structure):
    _fields_ = [(n, C.c_int32) for n in (
        "n_games", "height", "width", "n_players", "team_size", "n_cities", "city_army_lo",
        "city_army_hi", "spawn_dmin", "spawn_dmax", "spawn_exact", "max_turns", "auto_reset")] + [
        (n, C.c_uint32) for n in ("rule_flags", "game_id_base", "mountain_thr")] + [("seed", C.c_uint64)] + [
        (n, C.c_int32) for n in ("map_mode", "n_cities_max", "play_min", "castle_radius")]


class GenPolicy(C.Structure):
    _fields_ = [(n, C.c_uint32) for n in ("pass_thr", "half_thr", "bias_thr")]


# name -> (torch dtype name, shape builder(N, P, S, K))
BUFFERS = [
    ("army", "int16", lambda N, P, S, K: (N, S)),
    ("owner", "int8", lambda N, P, S, K: (N, S)),
    ("terrain", "int8", lambda N, P, S, K: (N, S)),
    ("turn", "int32", lambda N, P, S, K: (N,)),
    ("episode", "int32", lambda N, P, S, K: (N,)),            # bits of uint32
    ("alive", "uint8", lambda N, P, S, K: (N,)),
    ("general_cell", "int16", lambda N, P, S, K: (N, P)),
    ("land", "int32", lambda N, P, S, K: (N, P)),
    ("army_total", "int32", lambda N, P, S, K: (N, P)),
    ("reward", "int8", lambda N, P, S, K: (K, N, P)),
    ("done", "uint8", lambda N, P, S, K: (K, N)),
    ("winner", "int8", lambda N, P, S, K: (K, N)),
    ("obs_army", "int16", lambda N, P, S, K: (K, N, P, S)),
    ("obs_owner", "int8", lambda N, P, S, K: (K, N, P, S)),
    ("obs_terrain", "int8", lambda N, P, S, K: (K, N, P, S)),
    ("obs_vis", "uint8", lambda N, P, S, K: (K, N, P, S)),
    ("episodes_done", "int32", lambda N, P, S, K: (N,)),      # bits of uint32
    ("wins", "int32", lambda N, P, S, K: (N, P)),
    ("truncations", "int32", lambda N, P, S, K: (N,)),
    ("sat_events", "int32", lambda N, P, S, K: (N,)),
    ("obs_digest", "int64", lambda N, P, S, K: (N,)),         # bits of uint64
    ("actions_out", "int32", lambda N, P, S, K: (K, N, P)),
    ("bitboards", "int32", lambda N, P, S, K: (N, P + 3, (-(-S // 32) + 7) // 8 * 8)),   # bits of uint32
    ("obs_packed", "uint8", lambda N, P, S, K: (K, N, P, S)),
    ("score_hist", "int32", lambda N, P, S, K: (N, 512, 2 * P)),
    ("step_epoch", "int32", lambda N, P, S, K: (2, (N + 3) // 4)),                      # bits of uint32
    ("play_size", "int8", lambda N, P, S, K: (N, 2)),
    ("stack_cache", "int32", lambda N, P, S, K: (N, P + 1)),                             # bits of uint32
    ("invalid_actions", "int32", lambda N, P, S, K: (N,)),                               # bits of uint32
]


class GenBuffers(C.Structure):
    _fields_ = [(n, C.c_void_p) for n, _, _ in BUFFERS]


class GenSizes(C.Structure):
    _fields_ = ([("plane_stride", C.c_int32), ("alignment", C.c_int32)] + [(n, C.c_size_t) for n, _, _ in BUFFERS]
                + [("bitboard_row_words", C.c_int32)])


FEAT_CHANNELS = 38
# gen_feat_buffers: name -> (torch dtype name, shape builder(N, P, S))
FEAT_BUFFERS = [
    ("feat", "float32", lambda N, P, S: (N, P, FEAT_CHANNELS, S)),
    ("mem_bits", "uint8", lambda N, P, S: (N, P, S)),
    ("last_army", "int16", lambda N, P, S: (N, P, S)),
    ("last_seen", "int32", lambda N, P, S: (N, P, S)),
    ("hist", "int16", lambda N, P, S: (N, P, 8, 2, S)),
    ("feat_bf16", "bfloat16", lambda N, P, S: (N, P, FEAT_CHANNELS, S)),
]


class GenFeatBuffers(C.Structure):
    _fields_ = [(n, C.c_void_p) for n, _, _ in FEAT_BUFFERS]


class GenFeatSizes(C.Structure):
    _fields_ = ([("channels", C.c_int32), ("plane_stride", C.c_int32)] + [(n, C.c_size_t) for n, _, _ in FEAT_BUFFERS]
                + [("hist_windows", C.c_size_t)])


_lib = None


def load_library(path=None):
    """dlopen libgenerals.so and declare the signatures.  Raises if it has not been built."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    path = path or LIB_PATH
    if not os.path.exists(path):
        raise GenError(f"{path} is missing: build it with `python -m paper_2606_23348_b200.build` "
                       "(hand-written sm_100a kernels; there is no CPU fallback)")
    lib = C.CDLL(path)
    env_p = C.c_void_p
    lib.gen_query_sizes.argtypes = [C.POINTER(GenConfig), C.c_int32, C.POINTER(GenSizes)]
    lib.gen_init.argtypes = [C.POINTER(GenConfig), C.POINTER(env_p)]
    lib.gen_set_policy.argtypes = [env_p, C.POINTER(GenPolicy)]
    lib.gen_set_spawn.argtypes = [env_p, C.c_int32, C.c_int32, C.c_int32]
    lib.gen_set_spawn.restype = C.c_int
    lib.gen_global_step.argtypes = [env_p]
    lib.gen_global_step.restype = C.c_uint32
    lib.gen_set_global_step.argtypes = [env_p, C.c_uint32]
    lib.gen_reset.argtypes = [env_p, C.POINTER(GenBuffers), C.c_uint32, C.c_void_p]
    lib.gen_step.argtypes = [env_p, C.POINTER(GenBuffers), C.c_void_p, C.c_void_p]
    lib.gen_step_noalloc.argtypes = [env_p, C.POINTER(GenBuffers), C.c_void_p, C.c_void_p]
    lib.gen_step_noalloc.restype = C.c_int
    lib.gen_rollout.argtypes = [env_p, C.POINTER(GenBuffers), C.c_int32, C.c_uint32, C.c_void_p]
    lib.gen_observe.argtypes = [env_p, C.POINTER(GenBuffers), C.c_void_p]
    lib.gen_sample.argtypes = [env_p, C.POINTER(GenBuffers), C.c_void_p, C.c_void_p]
    lib.gen_step_host.argtypes = [env_p, C.POINTER(GenBuffers), C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
    lib.gen_step_host_async.argtypes = [env_p, C.POINTER(GenBuffers), C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
    lib.gen_host_wait.argtypes = [env_p, C.c_int32]
    lib.gen_forget_host_buffers.argtypes = [env_p]
    for name in ("gen_step_host_async", "gen_host_wait", "gen_forget_host_buffers"):
        getattr(lib, name).restype = C.c_int
    lib.gen_query_feat_sizes.argtypes = [C.POINTER(GenConfig), C.POINTER(GenFeatSizes)]
    lib.gen_features.argtypes = [env_p, C.POINTER(GenBuffers), C.POINTER(GenFeatBuffers), C.c_void_p]
    lib.gen_history_windows.argtypes = [env_p, C.POINTER(GenBuffers), C.c_void_p, C.c_void_p]
    lib.gen_history_windows.restype = C.c_int
    lib.gen_set_launch.argtypes = [env_p, C.c_int32]
    lib.gen_set_generic.argtypes = [env_p, C.c_int32, C.c_int32]
    lib.gen_set_chaining.argtypes = [env_p, C.c_int32]
    lib.gen_last_variant.argtypes = [env_p, C.POINTER(C.c_int32), C.POINTER(C.c_int32)]
    lib.gen_last_variant.restype = C.c_int32
    lib.gen_launch_count.argtypes = [env_p]
    lib.gen_launch_count.restype = C.c_uint64
    lib.gen_last_cuda_error.argtypes = [env_p]
    lib.gen_destroy.argtypes = [env_p]
    lib.gen_destroy.restype = None
    lib.gen_error_string.argtypes = [C.c_int]
    lib.gen_error_string.restype = C.c_char_p
    lib.gen_version.restype = C.c_char_p
    for name in ("gen_query_sizes", "gen_init", "gen_set_policy", "gen_set_global_step", "gen_reset",
                 "gen_step", "gen_rollout", "gen_observe", "gen_sample", "gen_step_host", "gen_set_launch",
                 "gen_set_generic", "gen_set_chaining", "gen_last_cuda_error", "gen_query_feat_sizes", "gen_features"):
        getattr(lib, name).restype = C.c_int
    if path == LIB_PATH:
        _lib = lib
    return lib


_CFG_KEYS = [n for n, _ in GenConfig._fields_]
_POLICY_KEYS = ("pass_thr", "half_thr", "bias_thr")


def make_config(cfg):
    """dict -> GenConfig; the policy thresholds (pass_thr / half_thr / bias_thr) are split off."""
    c = GenConfig()
    c.team_size = 1
    pol = {}
    for k, v in cfg.items():
        if k in _POLICY_KEYS:
            pol[k] = int(v)
        elif k in _CFG_KEYS:
            setattr(c, k, int(v))
        else:
            raise KeyError(f"unknown config key {k!r}")
    return c, pol


class GeneralsEnv:
    """N games on one GPU.  Owns the torch tensors the library works on.

    cfg: dict with the gen_config keys plus optional pass_thr / half_thr / bias_thr.
    k_slots > 1 sizes the output buffers for rollout(K, OBS_EVERY_STEP).
    """

    def __init__(self, cfg, device="cuda:0", k_slots=1, digest=True, actions_out=True, bitboards=True,
                 packed=False, history=False, chain=True, stack_cache=True):
        import torch
        self.torch = torch
        self.lib = load_library()
        if not torch.cuda.is_available():
            raise GenError("no CUDA device: the Generals.io step runs only on the GPU (no CPU fallback)")
        self.cfg, pol = make_config(cfg)
        self.device = torch.device(device)
        self.N, self.P, self.H, self.W = self.cfg.n_games, self.cfg.n_players, self.cfg.height, self.cfg.width
        self.HW = self.H * self.W
        self.K = int(k_slots)
        sizes = GenSizes()
        self._check(self.lib.gen_query_sizes(C.byref(self.cfg), self.K, C.byref(sizes)))
        self.S = sizes.plane_stride
        self._env = C.c_void_p()
        self._check(self.lib.gen_init(C.byref(self.cfg), C.byref(self._env)))
        self.bufs = GenBuffers()
        self.tensors = {}
        for name, dt, shape in BUFFERS:
            if ((name == "obs_digest" and not digest) or (name == "actions_out" and not actions_out)
                    or (name == "bitboards" and not bitboards) or (name == "obs_packed" and not packed) or (name == "score_hist" and not history) or (name == "step_epoch" and not chain) or (name == "stack_cache" and not stack_cache)
                    or (packed and name in ("obs_owner", "obs_terrain", "obs_vis"))):
                setattr(self.bufs, name, None)
                continue
            t = torch.zeros(shape(self.N, self.P, self.S, self.K), dtype=getattr(torch, dt), device=self.device)
            assert t.numel() * t.element_size() == getattr(sizes, name), name
            self.tensors[name] = t
            setattr(self, name, t)
            setattr(self.bufs, name, t.data_ptr() if t.numel() else None)
        if self.N == 0:
            for name, _, _ in BUFFERS:                     # any aligned non-NULL value passes validation
                if name in self.tensors:
                    setattr(self.bufs, name, 16)
        self._bufs_ref = C.byref(self.bufs)
        self.set_policy(**pol)

    # ------------------------------------------------------------------ plumbing
    def _check(self, code):
        if code != 0:
            msg = self.lib.gen_error_string(code).decode()
            cuda = self.lib.gen_last_cuda_error(self._env) if getattr(self, "_env", None) else 0
            raise GenError(f"generals: {msg} (code {code}, cuda error {cuda})")

    def _stream(self, stream=None):
        if stream is not None:
            return C.c_void_p(stream.cuda_stream)
        raw = getattr(self.torch._C, "_cuda_getCurrentRawStream", None)      # the current stream, without the wrapper
        if raw is not None:
            return C.c_void_p(raw(self.device.index if self.device.index is not None else self.torch.cuda.current_device()))
        return C.c_void_p(self.torch.cuda.current_stream(self.device).cuda_stream)

    def close(self):
        if getattr(self, "_env", None):
            self.lib.gen_destroy(self._env)
            self._env = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ------------------------------------------------------------------ the C ABI, same names
    def set_policy(self, pass_thr=0, half_thr=1 << 31, bias_thr=0):
        p = GenPolicy(int(pass_thr), int(half_thr), int(bias_thr))
        self._check(self.lib.gen_set_policy(self._env, C.byref(p)))

    def set_spawn(self, spawn_dmin, spawn_dmax=0, spawn_exact=0):
        """The spawn-distance curriculum: the window of the boards generated from now on."""
        self._check(self.lib.gen_set_spawn(self._env, int(spawn_dmin), int(spawn_dmax), int(spawn_exact)))
        self.cfg.spawn_dmin, self.cfg.spawn_dmax, self.cfg.spawn_exact = int(spawn_dmin), int(spawn_dmax), int(spawn_exact)

    @property
    def global_step(self):
        return int(self.lib.gen_global_step(self._env))

    @global_step.setter
    def global_step(self, v):
        self._check(self.lib.gen_set_global_step(self._env, int(v)))

    def set_launch(self, games_per_cta):
        self._check(self.lib.gen_set_launch(self._env, int(games_per_cta)))

    def set_generic(self, force_generic=True, force_staged=False):
        """Test hooks: never launch a board-specialised / the register-resident kernel (force_staged=-1:
        launch the register-resident kernel wherever it can serve, also for more than 4 players)."""
        self._check(self.lib.gen_set_generic(self._env, 1 if force_generic else 0, int(force_staged)))

    def set_chaining(self, enabled=True):
        """Launch chaining through step_epoch (see include/generals.h); off = every step waits for the whole grid."""
        self._check(self.lib.gen_set_chaining(self._env, 1 if enabled else 0))

    @property
    def last_launch_specialised(self):
        """True when the last launch used a kernel compiled for this exact board size and mode."""
        flag, rr = C.c_int32(0), C.c_int32(0)
        self.lib.gen_last_variant(self._env, C.byref(flag), C.byref(rr))
        return bool(flag.value)

    @property
    def last_launch_register_resident(self):
        """True when the last launch was the register-resident per-step kernel (generals_step.cuh)."""
        flag, rr = C.c_int32(0), C.c_int32(0)
        self.lib.gen_last_variant(self._env, C.byref(flag), C.byref(rr))
        return bool(rr.value)

    @property
    def launch_count(self):
        return int(self.lib.gen_launch_count(self._env))

    def reset(self, keep_episode=False, stream=None):
        self._check(self.lib.gen_reset(self._env, C.byref(self.bufs), GEN_KEEP_EPISODE if keep_episode else 0,
                                       self._stream(stream)))

    def step(self, actions=None, stream=None):
        """actions: int32 CUDA tensor [N][P] of flat action indices, or None for the built-in sampler."""
        ptr = None
        if actions is not None:
            assert actions.is_cuda and actions.dtype == self.torch.int32 and actions.is_contiguous()
            assert actions.numel() == self.N * self.P
            ptr = C.c_void_p(actions.data_ptr())
        code = self.lib.gen_step(self._env, self._bufs_ref, ptr, self._stream(stream))
        if code != 0:
            self._check(code)

    def step_noalloc(self, actions=None, stream=None):
        """gen_step_noalloc: step() for callers that cannot allocate device memory -- the bitboard cache comes from a
        fixed 8 MiB array inside the library (see include/generals.h for who needs this, the size limit and the rule
        that such calls must not overlap on the GPU).  Build the env with bitboards=False, digest=False."""
        ptr = None
        if actions is not None:
            assert actions.is_cuda and actions.dtype == self.torch.int32 and actions.is_contiguous()
            assert actions.numel() == self.N * self.P
            ptr = C.c_void_p(actions.data_ptr())
        self._check(self.lib.gen_step_noalloc(self._env, self._bufs_ref, ptr, self._stream(stream)))

    def rollout(self, K, obs_mode=OBS_DIGEST, stream=None):
        if obs_mode == OBS_EVERY_STEP and K > self.K:
            raise GenError(f"rollout(K={K}, OBS_EVERY_STEP) needs k_slots >= {K}, have {self.K}")
        self._check(self.lib.gen_rollout(self._env, C.byref(self.bufs), int(K), int(obs_mode), self._stream(stream)))

    def observe(self, stream=None):
        self._check(self.lib.gen_observe(self._env, C.byref(self.bufs), self._stream(stream)))

    def sample(self, out=None, stream=None):
        if out is None:
            out = self.torch.zeros((self.N, self.P), dtype=self.torch.int32, device=self.device)
        self._check(self.lib.gen_sample(self._env, C.byref(self.bufs), C.c_void_p(out.data_ptr()), self._stream(stream)))
        return out

    def features(self, stream=None, bf16=False):
        """NEXT-1 (R35): fold the current turn into each player's memory and return feat, a float32 CUDA tensor
        [N][P][38][S] (bf16=True: a bfloat16 tensor, R37; the choice is made at the first call).  Call once per turn
        (after reset and after every step).  More than two players: reading R38."""
        if not hasattr(self, "feat_bufs"):
            sizes = GenFeatSizes()
            self._check(self.lib.gen_query_feat_sizes(C.byref(self.cfg), C.byref(sizes)))
            self.feat_bufs = GenFeatBuffers()
            self.feat_tensors = {}
            for name, dt, shape in FEAT_BUFFERS:
                if name == ("feat" if bf16 else "feat_bf16"):
                    setattr(self.feat_bufs, name, None)
                    continue
                t = self.torch.zeros(shape(self.N, self.P, self.S), dtype=getattr(self.torch, dt), device=self.device)
                assert t.numel() * t.element_size() == getattr(sizes, name), name
                self.feat_tensors[name] = t
                setattr(self.feat_bufs, name, t.data_ptr() if t.numel() else 16)
            self.feat = self.feat_tensors["feat_bf16" if bf16 else "feat"]
        self._check(self.lib.gen_features(self._env, C.byref(self.bufs), C.byref(self.feat_bufs), self._stream(stream)))
        return self.feat

    def history_windows(self, out=None, stream=None):
        """NEXT-2 (R39): int32 CUDA tensor [N][P][2][512] -- the enemies' army (0) and land (1) totals over the
        last 512 turns of the current episode, oldest first, 0 before its first turn.  Needs history=True."""
        if out is None:
            if not hasattr(self, "_windows"):
                self._windows = self.torch.zeros((self.N, self.P, 2, 512), dtype=self.torch.int32, device=self.device)
            out = self._windows
        self._check(self.lib.gen_history_windows(self._env, C.byref(self.bufs), C.c_void_p(out.data_ptr() if out.numel() else 16),
                                                 self._stream(stream)))
        return out

    def step_host(self, h_actions=None, h_reward=None, h_done=None, stream=None):
        """End to end through host buffers (pinned CPU tensors); synchronises the stream."""
        ptr = lambda t: None if t is None else C.c_void_p(t.data_ptr())   # noqa: E731
        for t in (h_actions, h_reward, h_done):
            assert t is None or (not t.is_cuda and t.is_contiguous())
        self._check(self.lib.gen_step_host(self._env, C.byref(self.bufs), ptr(h_actions), ptr(h_reward),
                                           ptr(h_done), self._stream(stream)))

    def step_host_async(self, h_actions=None, h_reward=None, h_done=None, stream=None):
        """gen_step_host without the synchronisation; host_wait(lag) tells when a call's results have landed."""
        ptr = lambda t: None if t is None else C.c_void_p(t.data_ptr())   # noqa: E731
        code = self.lib.gen_step_host_async(self._env, self._bufs_ref, ptr(h_actions), ptr(h_reward), ptr(h_done),
                                            self._stream(stream))
        if code != 0:
            self._check(code)

    def host_wait(self, lag=0):
        code = self.lib.gen_host_wait(self._env, int(lag))
        if code != 0:
            self._check(code)

    def forget_host_buffers(self):
        self._check(self.lib.gen_forget_host_buffers(self._env))

    # ------------------------------------------------------------------ helpers
    def field(self, name, slot=0):
        """numpy view of a buffer (unsigned where the C type is unsigned); slot 0 of [K]-strided ones."""
        import numpy as np
        t = self.tensors[name]
        if name in ("reward", "done", "winner", "obs_army", "obs_owner", "obs_terrain", "obs_vis", "actions_out",
                    "obs_packed"):
            t = t[slot]
        a = t.cpu().numpy()
        if name in ("episode", "episodes_done", "wins", "truncations", "sat_events", "invalid_actions"):
            a = a.view(np.uint32)
        elif name == "obs_digest":
            a = a.view(np.uint64)
        return a
