// generals_features.h -- launch parameters of k_features (generals_features.cu), shared with generals_api.cu.
#pragma once
#include <cuda_runtime.h>
#include <cstdint>

namespace gen {

struct FeatParams {
    int N, H, W, HW, S;
    int P, team_size;            // players, team size (1v1: 2, 1: the tuned kernel; else R38's)
    int G;                       // games per CTA (2 * S / 4 threads each)
    int force_generic;           // never launch a board-specialised instantiation (tests)
    const int16_t *army;         // state planes and scalars of gen_buffers (read only)
    const int8_t *owner;
    const int8_t *terrain;
    const int32_t *turn;
    const int32_t *land;
    const int32_t *army_total;
    const int8_t *play_size;     // [N][2] playable rows, columns (or NULL / 0: the full board)
    int bf16;                    // feat points at bfloat16 (R37) instead of float
    void *feat;                  // gen_feat_buffers: feat or feat_bf16
    uint8_t *mem_bits;
    int16_t *last_army;
    int32_t *last_seen;
    int16_t *hist;
};

cudaError_t launch_features(const FeatParams &fp, cudaStream_t stream);

// gen_history_windows (R39): ring = gen_buffers.score_hist [N][512][2P], win = int32 [N][P][2][512]
cudaError_t launch_history_windows(const int32_t *ring, const int32_t *turn, int32_t *win, int N, int P, int team_size,
                                   cudaStream_t stream);

}  // namespace gen
