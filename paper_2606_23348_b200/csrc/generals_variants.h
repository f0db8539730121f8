// generals_variants.h -- the list of kernel instantiations of libgenerals.so.
// One translation unit per variant (generals_variant.cu compiled with -DGEN_VARIANT_ID=n) so that the
// build compiles them in parallel; generals_api.cu picks one per launch from this table.
#pragma once
#include <cuda_runtime.h>

#include "generals_kernels.cuh"

namespace gen {

constexpr uint32_t FF_STEP = F_OBS_PLANES | F_K1;                // gen_step without a digest buffer
constexpr uint32_t FF_ROLL_DIGEST = F_OBS_PLANES | F_DIGEST;     // gen_rollout(K, GEN_OBS_DIGEST)

//  X(id, NP, H, W, flags)
#define GEN_VARIANTS(X)            \
    X(0, 2, 0, 0, F_RUNTIME)       \
    X(1, 4, 0, 0, F_RUNTIME)       \
    X(2, 8, 0, 0, F_RUNTIME)       \
    X(3, 2, 24, 24, FF_STEP)       \
    X(4, 2, 24, 24, FF_ROLL_DIGEST)\
    X(5, 2, 8, 8, FF_STEP)         \
    X(6, 4, 32, 32, FF_STEP)       \
    X(7, 8, 32, 32, FF_STEP)
constexpr int N_VARIANTS = 8;

struct Variant {
    int np, h, w;      // h == 0: any board with n_players <= np
    uint32_t ff;       // F_RUNTIME: any mode
    cudaError_t (*launch)(const KParams &, int grid, int block, size_t smem, cudaStream_t);
};

#define GEN_DECLARE(id, np, h, w, ff) \
    cudaError_t launch_variant_##id(const KParams &, int grid, int block, size_t smem, cudaStream_t);
GEN_VARIANTS(GEN_DECLARE)
#undef GEN_DECLARE

constexpr size_t kMaxSmem = 200 * 1024;

}  // namespace gen
