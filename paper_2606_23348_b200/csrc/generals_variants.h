// generals_variants.h -- the list of kernel instantiations of libgenerals.so.
// One translation unit per variant (generals_variant.cu compiled with -DGEN_VARIANT_ID=n) so that the
// build compiles them in parallel; generals_api.cu picks one per launch from this table.
//   kind 0: the STAGED kernel k_generals (generals_kernels.cuh): planes resident in shared memory; serves
//           every call (reset, observe, sample, step, K-step rollout, digest).
//   kind 2 / 3: kind 0 / 1 with the official map generator (see the end of the table).
//   kind 1: the REGISTER-RESIDENT per-step kernel k_step (generals_step.cuh): gen_step when the caller
//           provides the bitboard cache and no digest buffer.
#pragma once
#include <cuda_runtime.h>

#include "generals_step.cuh"

namespace gen {

// variant 12: gen_step on the staged kernel at 24x24 1v1 (callers without the bitboard cache)
constexpr uint32_t FF_ROLL_DIGEST = F_OBS_PLANES | F_DIGEST;     // gen_rollout(K, GEN_OBS_DIGEST)

//  X(id, kind, NP, H, W, flags (kind 0) or 0, max threads per CTA, min CTAs per SM (kind 1))
#define GEN_VARIANTS(X)                          \
    X(0, 0, 2, 0, 0, F_RUNTIME, 256, 1)          \
    X(1, 0, 4, 0, 0, F_RUNTIME, 256, 1)          \
    X(2, 0, 8, 0, 0, F_RUNTIME, 256, 1)          \
    X(3, 0, 2, 24, 24, FF_ROLL_DIGEST, 256, 1)   \
    X(4, 1, 2, 0, 0, 0, 256, 2)                  \
    X(5, 1, 4, 0, 0, 0, 256, 2)                  \
    X(6, 1, 8, 0, 0, 0, 256, 2)                  \
    X(7, 1, 2, 24, 24, 0, 64, 14)                \
    X(8, 1, 2, 8, 8, 0, 64, 16)                  \
    X(9, 1, 4, 32, 32, 0, 64, 8)                 \
    X(10, 1, 8, 32, 32, 0, 64, 6)                \
    X(11, 1, 2, 24, 24, 0, 64, 10)               \
    X(12, 0, 2, 24, 24, F_OBS_PLANES, 256, 1)    \
    X(13, 3, 2, 23, 23, 0, 64, 14)               \
    X(14, 3, 2, 23, 23, 0, 64, 10)               \
    X(15, 2, 2, 0, 0, F_RUNTIME, 256, 1)         \
    X(16, 3, 2, 0, 0, 0, 256, 2)                 \
    X(17, 1, 2, 24, 24, 0, 64, 12)               \
    X(18, 1, 2, 24, 24, 1, 64, 14)               \
    X(19, 1, 2, 24, 24, 1, 64, 12)               \
    X(20, 1, 2, 24, 24, 1, 64, 10)               \
    X(21, 0, 8, 32, 32, F_OBS_PLANES, 256, 1)    \
    X(22, 0, 2, 24, 24, F_OBS_PLANES | F_OBS_EVERY, 256, 1)  \
    X(23, 0, 2, 24, 24, F_RESET | F_OBS_PLANES, 256, 1)      \
    X(24, 2, 2, 23, 23, F_RESET | F_OBS_PLANES, 256, 1)      \
    X(25, 0, 4, 32, 32, F_RESET | F_OBS_PLANES, 256, 1)      \
    X(26, 0, 8, 32, 32, F_RESET | F_OBS_PLANES, 256, 1)
constexpr int N_VARIANTS = 27;
// Variant 21: gen_step of the 8-player free-for-all on 32x32 (BASELINE config 5b) on the staged kernel compiled for
// that board and mode (more than 4 players stay on the staged kernel, generals_api.cu): 83 -> 101 M env steps/s at
// 32,768 games (57 -> 69.5 % of the HBM copy peak).  The same for 2v2 (4, 32, 32) was tried and is slower than
// k_step<4,32,32> (175 M against 192 M), so it is not in the table.
// Variant 22: gen_rollout(K, GEN_OBS_EVERY_STEP) on 24x24 1v1 (the planes of every turn written): 698 -> 836-844 M env
// steps/s at 16,384 games, 811 -> 944-947 M at 262,144 (the generic kernel served this call before).
// Variant 23: gen_reset on 24x24 1v1 (synthetic generator + first observation): 108 -> 92 us for 16,384 boards,
// 196 -> 222 M maps/s at 262,144.  Variant 24: the same for the official generator on 23x23 (118 -> 132 M maps/s).
// Variants 25 / 26: gen_reset of config 5's boards (2v2: 691 -> 538 us, FFA-8: 1,516 -> 1,250 us for 32,768 boards).
// Variants 18-20: variants 7 / 17 / 11 for the biased policy (R25; BASELINE config 4): flags = 1 compiles the
// observation pass that also finds each player's largest owned stack and leaves it in gen_buffers.stack_cache.
// Kinds 2 / 3 are kinds 0 / 1 compiled with the official map generator (R36; gen_config.map_mode = 1, 1v1 only): the
// generator is a template flag, not a runtime branch, so that the kernels of BASELINE's configs are exactly what they
// were without it.  Variants 13 and 14: the paper's own board ("up to 23x23"; workload official_23x23) under
// the same two register budgets as 7 and 11; 15 / 16: any other 1v1 board.
// Variant 17: the same kernel once more at 80 registers / 12 CTAs per SM, the best of the three for batches of more than
// one wave whose launches still chain (measured: +3-5 % over variant 11 from 24,576 to 131,072 games).
// Variants 7 and 11 are the same kernel under two register budgets: 72 registers (14 CTAs of 8 games per SM:
// a batch of up to 16,576 games -- BASELINE config 2's 16,384 -- is resident in ONE wave) and 96 registers (10 CTAs
// per SM, no spills: faster per wave, the choice whenever the batch fits 10 CTAs per SM or needs several waves anyway).

struct Variant {
    int kind, np, h, w;  // h == 0: any board with n_players <= np
    uint32_t ff;         // kind 0: F_RUNTIME = any mode, else the exact mode
    int max_threads;     // largest CTA this instantiation may be launched with
    int min_ctas;        // resident CTAs per SM its register budget allows (launch bounds)
    cudaError_t (*launch)(const KParams &, int grid, int block, size_t smem, cudaStream_t);
};

#define GEN_DECLARE(id, kind, np, h, w, ff, maxt, minb) \
    cudaError_t launch_variant_##id(const KParams &, int grid, int block, size_t smem, cudaStream_t);
GEN_VARIANTS(GEN_DECLARE)
#undef GEN_DECLARE

constexpr size_t kMaxSmem = 200 * 1024;

}  // namespace gen
