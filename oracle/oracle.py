"""ctypes front end of the CPU oracle (oracle/generals_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, bench.py's cpu_baseline /
``--impl reference`` leg and ``__graft_entry__.smoke()`` may import this module.
It shares nothing with ``paper_2606_23348_b200`` (no import in either direction).
All state lives in numpy arrays owned by :class:`Oracle`.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "generals_oracle.c")
_LIB = os.path.join(_HERE, "libgenerals_oracle.so")

T_PLAIN, T_MOUNTAIN, T_CITY, T_GENERAL, T_FOG = 0, 1, 2, 3, 4
OWNER_NEUTRAL, OWNER_FOG = -1, -2
RULE_TICK_PLAIN_ONLY, RULE_CAPTURE_HALF_FLOOR, RULE_ROTATE_PRIORITY = 1, 2, 4
OBS_DIGEST, OBS_EVERY_STEP, OBS_NONE = 0, 1, 2


def build(force=False):
    """Compile the oracle with gcc (plain C99, -O2). Building the checker is not using it."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-std=c99", "-O2", "-Wall", "-Wextra", "-fPIC", "-shared",
                               "-o", _LIB, _SRC, "-lm"])
    return _LIB


class OrcConfig(C.Structure):
    _fields_ = [(n, C.c_int32) for n in (
        "n_games", "height", "width", "n_players", "team_size", "n_cities", "city_army_lo",
        "city_army_hi", "spawn_dmin", "spawn_dmax", "spawn_exact", "max_turns", "auto_reset")] + [
        (n, C.c_uint32) for n in ("rule_flags", "game_id_base", "mountain_thr", "pass_thr", "half_thr",
                                  "bias_thr", "pad_")] + [("seed", C.c_uint64)] + [
        (n, C.c_int32) for n in ("map_mode", "n_cities_max", "play_min", "castle_radius")]


_BUF_FIELDS = [
    ("army", np.int16), ("owner", np.int8), ("terrain", np.int8), ("turn", np.int32),
    ("episode", np.uint32), ("alive", np.uint8), ("general_cell", np.int16), ("land", np.int32),
    ("army_total", np.int32), ("reward", np.int8), ("done", np.uint8), ("winner", np.int8),
    ("obs_army", np.int16), ("obs_owner", np.int8), ("obs_terrain", np.int8), ("obs_vis", np.uint8),
    ("episodes_done", np.uint32), ("wins", np.uint32), ("truncations", np.uint32),
    ("sat_events", np.uint32), ("obs_digest", np.uint64), ("obs_packed", np.uint8),
    ("score_hist", np.int32), ("play_size", np.int8), ("invalid_actions", np.uint32),
]


class OrcFeatState(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in ("bits", "last_army", "last_turn", "hist")]


class OrcBuffers(C.Structure):
    _fields_ = [(n, C.c_void_p) for n, _ in _BUF_FIELDS]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_philox4x32_10.argtypes = [C.POINTER(C.c_uint32)] * 3
        _lib.orc_philox4x32_10.restype = None
        _lib.orc_mix64.argtypes = [C.c_uint64]
        _lib.orc_mix64.restype = C.c_uint64
        _lib.orc_digest_key.argtypes = [C.c_int32]
        _lib.orc_digest_key.restype = C.c_uint64
        _lib.orc_plane_stride.argtypes = [C.POINTER(OrcConfig)]
        _lib.orc_reset.argtypes = [C.POINTER(OrcConfig), C.POINTER(OrcBuffers)]
        _lib.orc_sample.argtypes = [C.POINTER(OrcConfig), C.POINTER(OrcBuffers), C.c_uint32, C.c_void_p]
        _lib.orc_step.argtypes = [C.POINTER(OrcConfig), C.POINTER(OrcBuffers), C.c_void_p, C.c_uint32,
                                  C.c_void_p]
        _lib.orc_rollout.argtypes = [C.POINTER(OrcConfig), C.POINTER(OrcBuffers), C.c_int32, C.c_uint32,
                                     C.c_int32]
        _lib.orc_observe.argtypes = [C.POINTER(OrcConfig), C.POINTER(OrcBuffers)]
        _lib.orc_features.argtypes = [C.POINTER(OrcConfig), C.POINTER(OrcBuffers), C.POINTER(OrcFeatState), C.c_void_p]
        _lib.orc_history_windows.argtypes = [C.POINTER(OrcConfig), C.POINTER(OrcBuffers), C.c_void_p]
        _lib.orc_features_bf16.argtypes = [C.POINTER(OrcConfig), C.POINTER(OrcBuffers), C.POINTER(OrcFeatState),
                                           C.c_void_p, C.c_void_p]
    return _lib


def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*ctr)
    k = (C.c_uint32 * 2)(*key)
    o = (C.c_uint32 * 4)()
    lib().orc_philox4x32_10(c, k, o)
    return tuple(int(x) for x in o)


def mix64(z):
    return int(lib().orc_mix64(C.c_uint64(z)))


def digest_key(c):
    return int(lib().orc_digest_key(c))


_CFG_KEYS = {n for n, _ in OrcConfig._fields_} - {"pad_"}


class Oracle:
    """N games held in numpy arrays shaped like the device buffers of the CUDA path.

    ``cfg`` is a plain dict with the keys of ``orc_config`` (missing keys default to 0,
    ``team_size`` to 1); ``every_step_K`` > 0 sizes the obs / reward / done / winner
    buffers for ``rollout(K, OBS_EVERY_STEP)``.
    """

    def __init__(self, cfg, every_step_K=0, digest=True):
        unknown = set(cfg) - _CFG_KEYS
        if unknown:
            raise KeyError(f"unknown config keys {sorted(unknown)}")
        self.cfg = OrcConfig()
        self.cfg.team_size = 1
        for k, v in cfg.items():
            setattr(self.cfg, k, int(v))
        c = self.cfg
        self.N, self.P, self.H, self.W = c.n_games, c.n_players, c.height, c.width
        self.HW = self.H * self.W
        self.S = int(lib().orc_plane_stride(C.byref(c)))
        N, P, S = self.N, self.P, self.S
        Kb = max(1, every_step_K)
        shapes = {
            "army": (N, S), "owner": (N, S), "terrain": (N, S), "turn": (N,), "episode": (N,),
            "alive": (N,), "general_cell": (N, P), "land": (N, P), "army_total": (N, P),
            "reward": (Kb, N, P), "done": (Kb, N), "winner": (Kb, N),
            "obs_army": (Kb, N, P, S), "obs_owner": (Kb, N, P, S), "obs_terrain": (Kb, N, P, S),
            "obs_vis": (Kb, N, P, S), "episodes_done": (N,), "wins": (N, P), "truncations": (N,),
            "sat_events": (N,), "obs_digest": (N,), "obs_packed": (Kb, N, P, S),
            "score_hist": (N, 512, 2 * P), "play_size": (N, 2), "invalid_actions": (N,),
        }
        self.bufs = OrcBuffers()
        for name, dt in _BUF_FIELDS:
            a = np.zeros(shapes[name], dtype=dt)
            setattr(self, name, a)
            if name == "obs_digest" and not digest:
                setattr(self.bufs, name, None)
            else:
                setattr(self.bufs, name, a.ctypes.data)
        self.global_step = 0

    # views of slot 0 (the only slot unless every_step_K > 0)
    def field(self, name):
        a = getattr(self, name)
        return a[0] if name in ("reward", "done", "winner", "obs_army", "obs_owner", "obs_terrain",
                                "obs_vis", "obs_packed") else a

    def reset(self):
        lib().orc_reset(C.byref(self.cfg), C.byref(self.bufs))
        self.global_step = 0

    def sample(self):
        out = np.zeros((self.N, self.P), dtype=np.int32)
        lib().orc_sample(C.byref(self.cfg), C.byref(self.bufs), self.global_step, out.ctypes.data)
        return out

    def step(self, actions=None, want_actions=False):
        out = np.zeros((self.N, self.P), dtype=np.int32) if want_actions else None
        if actions is not None:
            actions = np.ascontiguousarray(actions, dtype=np.int32).reshape(self.N, self.P)
        lib().orc_step(C.byref(self.cfg), C.byref(self.bufs),
                       None if actions is None else actions.ctypes.data, self.global_step,
                       None if out is None else out.ctypes.data)
        self.global_step += 1
        return out

    def rollout(self, K, obs_mode=OBS_DIGEST):
        lib().orc_rollout(C.byref(self.cfg), C.byref(self.bufs), K, self.global_step, obs_mode)
        self.global_step += K

    def observe(self):
        lib().orc_observe(C.byref(self.cfg), C.byref(self.bufs))

    def features(self, bf16=False):
        """NEXT-1: fold the current turn into the per-episode memory and return feat[N][2][38][S] (float32; with
        bf16=True the bfloat16 bit patterns as uint16, R37).  Call once per turn (after reset and after every step)."""
        N, S, P = self.N, self.S, self.P
        if not hasattr(self, "feat"):
            self.feat = np.zeros((N, P, 38, S), dtype=np.float32)
            self._fm = dict(bits=np.zeros((N, P, 5, S), np.uint8), last_army=np.zeros((N, P, S), np.int16),
                            last_turn=np.full((N, P, S), -1, np.int32), hist=np.zeros((N, P, 2, 8, S), np.int16))
            self._fs = OrcFeatState(*[self._fm[k].ctypes.data for k in ("bits", "last_army", "last_turn", "hist")])
        if bf16:
            if not hasattr(self, "feat16"):
                self.feat16 = np.zeros((N, P, 38, S), dtype=np.uint16)
            rc = lib().orc_features_bf16(C.byref(self.cfg), C.byref(self.bufs), C.byref(self._fs),
                                         self.feat.ctypes.data, self.feat16.ctypes.data)
        else:
            rc = lib().orc_features(C.byref(self.cfg), C.byref(self.bufs), C.byref(self._fs), self.feat.ctypes.data)
        if rc != 0:
            raise ValueError("orc_features failed")
        return self.feat16 if bf16 else self.feat

    def history_windows(self):
        """NEXT-2 (R39): int32 [N][P][2][512] -- the enemies' army (0) and land (1) totals over the last 512
        turns of the current episode, oldest first, 0 before the episode's first turn."""
        win = np.zeros((self.N, self.P, 2, 512), dtype=np.int32)
        if lib().orc_history_windows(C.byref(self.cfg), C.byref(self.bufs), win.ctypes.data) != 0:
            raise ValueError("orc_history_windows failed")
        return win

    def set_policy(self, pass_thr=None, half_thr=None, bias_thr=None):
        for k, v in (("pass_thr", pass_thr), ("half_thr", half_thr), ("bias_thr", bias_thr)):
            if v is not None:
                setattr(self.cfg, k, int(v))

    def board_str(self, g=0):
        """ASCII dump of game g (debugging aid)."""
        rows = []
        for r in range(self.H):
            cells = []
            for c in range(self.W):
                i = r * self.W + c
                t, o, a = int(self.terrain[g, i]), int(self.owner[g, i]), int(self.army[g, i])
                sym = ".#CG"[t]
                cells.append(f"{sym}{'-' if o < 0 else o}{a:>3}")
            rows.append(" ".join(cells))
        return "\n".join(rows)
