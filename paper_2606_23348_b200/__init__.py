"""B200-native batched Generals.io environment step (arXiv 2606.23348, section IV).

`GeneralsEnv` is a thin binding over the C ABI of include/generals.h: torch provides device memory
and streams, every step of the path runs in the hand-written sm_100a kernels of csrc/.
"""
from .binding import (GEN_KEEP_EPISODE, OBS_DIGEST, OBS_EVERY_STEP, OBS_NONE, GenConfig, GeneralsEnv,
                      GenError, load_library)

__all__ = ["GeneralsEnv", "GenConfig", "GenError", "load_library", "OBS_DIGEST", "OBS_EVERY_STEP",
           "OBS_NONE", "GEN_KEEP_EPISODE"]
