"""In-tree build of the CUDA library (sm_100a only): `python -m paper_2606_23348_b200.build`.

nvcc cross-compiles without a GPU.  The kernel is one template; every instantiation listed in
csrc/generals_variants.h is its own translation unit (generals_variant.cu with -DGEN_VARIANT_ID=n),
compiled in parallel and linked with the host API into libgenerals.so, which sits next to this file,
is git-ignored and travels to the GPU box with the repo snapshot.
"""
import os
import re
import shutil
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libgenerals.so")
DEPS = [os.path.join(CSRC, f) for f in ("generals_api.cu", "generals_variant.cu", "generals_variants.h",
                                        "generals_kernels.cuh", "generals_step.cuh", "generals_features.cu",
                                        "generals_features.h", "generals_noalloc.cu")] + [os.path.join(ROOT, "include", "generals.h")]
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]


def nvcc_path():
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: the CUDA library cannot be built (there is no CPU fallback)")


def n_variants():
    with open(os.path.join(CSRC, "generals_variants.h")) as f:
        return int(re.search(r"N_VARIANTS\s*=\s*(\d+)", f.read()).group(1))


def build(force=False, verbose=False):
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in DEPS):
        return LIB
    os.makedirs(OBJ, exist_ok=True)
    base = [nvcc_path(), "-std=c++17", "-O3", *ARCH, "-lineinfo", "-Xcompiler", "-fPIC",
            "-I", os.path.join(ROOT, "include"), "-I", CSRC]
    base += os.environ.get("GEN_NVCC_FLAGS", "").split()      # development only (e.g. -DGEN_EXPERIMENT=...)
    if verbose:
        base += ["-Xptxas", "-v"]
    jobs = [(base + ["-c", os.path.join(CSRC, "generals_api.cu"), "-o", os.path.join(OBJ, "api.o")])]
    jobs.append(base + ["-c", os.path.join(CSRC, "generals_features.cu"), "-o", os.path.join(OBJ, "features.o")])
    jobs.append(base + ["-c", os.path.join(CSRC, "generals_noalloc.cu"), "-o", os.path.join(OBJ, "noalloc.o")])
    for i in range(n_variants()):
        jobs.append(base + [f"-DGEN_VARIANT_ID={i}", "-c", os.path.join(CSRC, "generals_variant.cu"),
                            "-o", os.path.join(OBJ, f"variant{i}.o")])

    def run(cmd):
        if verbose:
            print(" ".join(cmd), file=sys.stderr)
        subprocess.check_call(cmd)

    with ThreadPoolExecutor(max_workers=min(len(jobs), os.cpu_count() or 4)) as pool:
        list(pool.map(run, jobs))
    objs = [j[-1] for j in jobs]
    run([nvcc_path(), *ARCH, "-shared", "-o", LIB] + objs)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
