// generals_noalloc.cu -- gen_step_noalloc (include/generals.h): one turn on the register-resident per-step kernel
// for callers that cannot give the library a bitboard cache because they cannot allocate device memory.
//
// Who that is.  The fast per-step kernel (k_step, generals_step.cuh) needs gen_buffers.bitboards, 480 bytes per game
// of working memory at 24x24 that is neither an input nor a result of the step.  A normal caller gets it from
// cudaMalloc (or from torch) once and passes it in.  Some callers have no such option at the point where they step
// the games:
//   * an environment that runs as an operator inside somebody else's executor (a custom call of a compiled training
//     graph, a plug-in of an inference runtime): the executor owns all device memory, hands the operator its operands
//     and its results and no workspace, and calling the CUDA allocator behind its back is not allowed;
//   * a training process that has handed every byte of HBM to the learner's arena at start-up, so that a later
//     cudaMalloc simply fails;
//   * a latency-sensitive actor loop: cudaMalloc and cudaFree synchronise the device, which stalls every other stream
//     of the process for the duration of the call.
// For them the library carries the working memory itself: one file-scope device array of GEN_NOALLOC_SCRATCH_BYTES
// (8 MiB, enough for 17,476 games of 24x24 1v1) that exists on every GPU the library is loaded on, from load to
// process exit.  The call below rebuilds the cache rows in that array from the caller's planes with a small kernel of
// its own and then runs the ordinary gen_step with the array in the place of the caller's buffer.  Nothing here calls
// cudaMalloc, cudaFree or any routine that allocates.
//
// The array's NAME is usable in device code only.  In host code `g_noalloc_scratch` is a host-side shadow symbol: its
// address is not a device address, and a kernel handed that address faults (or, on a system where the GPU can reach
// host memory, quietly works on the wrong bytes).  The device address is asked for with cudaGetSymbolAddress once per
// device, with that device current, and that is the pointer the kernels receive.
#include <cuda_runtime.h>

#include <mutex>

#include "generals.h"

namespace gen {
// generals_api.cu: what this file needs of the opaque handle
const gen_config *env_config(const gen_env *env);
void env_count_launch(gen_env *env);
}  // namespace gen

namespace {

static __device__ __align__(256) unsigned char g_noalloc_scratch[GEN_NOALLOC_SCRATCH_BYTES];

constexpr int kMaxDevices = 64;
void *g_scratch_addr[kMaxDevices];  // device address of g_noalloc_scratch on device d; nullptr = not asked for yet
std::mutex g_setup_lock;

// Device address of the scratch array on the CURRENT device.  The first call on a device asks the runtime for it
// (this also makes the runtime load the module on that device, which is why that call belongs before any stream
// capture); later calls read the table.
cudaError_t scratch_on_current_device(void **out) {
    int dev = 0;
    if (cudaError_t e = cudaGetDevice(&dev); e != cudaSuccess) return e;
    std::lock_guard<std::mutex> hold(g_setup_lock);
    if (dev >= 0 && dev < kMaxDevices && g_scratch_addr[dev]) { *out = g_scratch_addr[dev]; return cudaSuccess; }
    void *p = nullptr;
    if (cudaError_t e = cudaGetSymbolAddress(&p, g_noalloc_scratch); e != cudaSuccess) return e;
    if (!p) return cudaErrorInvalidSymbol;
    if (dev >= 0 && dev < kMaxDevices) g_scratch_addr[dev] = p;
    *out = p;
    return cudaSuccess;
}

// The cache rows of gen_buffers.bitboards from the three planes, one warp per game: rows 0..P-1 "owned by player p",
// row P "army >= 2", row P+1 "city or general", row P+2 "mountain or off the board"; bit c & 31 of word c >> 5; BW
// words per row; everything past cell H*W reads 0 (1 in the last row).  Every word of the N games is written, so the
// step that follows never sees what an earlier call left in the array.
__global__ void __launch_bounds__(256) k_noalloc_rows(const int16_t *__restrict__ army, const int8_t *__restrict__ owner,
                                                      const int8_t *__restrict__ terrain, uint32_t *__restrict__ rows,
                                                      int N, int P, int HW, int S, int BW) {
    const int lane = (int)(threadIdx.x & 31u);
    const int g = (int)(blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5));
    if (g >= N) return;  // the whole warp leaves together
    const size_t base = (size_t)g * (size_t)S;
    uint32_t mine[7] = {0u, 0u, 0u, 0u, 0u, 0u, 0u};  // lane j keeps word j of each of the P + 3 <= 7 rows
    for (int j = 0; j < BW; ++j) {
        const int c = 32 * j + lane;
        const bool in = c < HW;
        int a = 0, o = -1, t = 1;
        if (in) { a = army[base + c]; o = owner[base + c]; t = terrain[base + c]; }
        uint32_t own[4];
#pragma unroll
        for (int p = 0; p < 4; ++p) own[p] = __ballot_sync(0xffffffffu, in && o == p);
        const uint32_t a2 = __ballot_sync(0xffffffffu, in && a >= 2);
        const uint32_t str = __ballot_sync(0xffffffffu, in && t >= 2);
        const uint32_t mtn = __ballot_sync(0xffffffffu, !in || t == 1);
        if (lane == j) {
#pragma unroll
            for (int r = 0; r < 7; ++r)
                mine[r] = r < P ? own[r < 4 ? r : 3] : (r == P ? a2 : (r == P + 1 ? str : mtn));
        }
    }
    uint32_t *dst = rows + (size_t)g * (size_t)(P + 3) * (size_t)BW;
#pragma unroll
    for (int r = 0; r < 7; ++r)
        if (r < P + 3 && lane < BW) dst[r * BW + lane] = mine[r];
}

bool aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

}  // namespace

extern "C" int gen_step_noalloc(gen_env *env, const gen_buffers *bufs, const int32_t *d_actions, void *cuda_stream) {
    if (!env || !bufs) return GEN_ERR_NULL;
    const gen_config *cfg = gen::env_config(env);
    const size_t N = (size_t)cfg->n_games, P = (size_t)cfg->n_players;
    const int HW = cfg->height * cfg->width, S = (HW + 15) / 16 * 16, BW = ((HW + 31) / 32 + 7) / 8 * 8;
    // the register-resident kernel serves up to four players and no digest buffer; anything else would run the staged
    // kernel, which needs no cache and therefore no scratch: plain gen_step with bitboards = NULL is the call for it
    if (P > 4 || bufs->obs_digest) return GEN_ERR_ARG;
    if (N * (P + 3) * (size_t)BW * 4u > (size_t)GEN_NOALLOC_SCRATCH_BYTES) return GEN_ERR_SIZE;
    // the three planes this file's own kernel reads; gen_step checks every buffer again
    if (!bufs->army || !bufs->owner || !bufs->terrain) return GEN_ERR_NULL;
    if (!aligned16(bufs->army) || !aligned16(bufs->owner) || !aligned16(bufs->terrain)) return GEN_ERR_ALIGN;
    gen_buffers b = *bufs;
    b.step_epoch = nullptr;   // no launch chaining: a chained step would not wait for the kernel that rebuilds the rows
    b.stack_cache = nullptr;  // the biased sampler scans the army plane
    if (N == 0) { b.bitboards = nullptr; return gen_step(env, &b, d_actions, cuda_stream); }
    void *scratch = nullptr;
    if (scratch_on_current_device(&scratch) != cudaSuccess) { (void)cudaGetLastError(); return GEN_ERR_CUDA; }
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    const int warps_per_cta = 8;
    const unsigned grid = (unsigned)((N + warps_per_cta - 1) / warps_per_cta);
    // a plain launch: it starts only when everything earlier in the stream -- also a previous call's step kernel, which
    // writes changed rows back into the array -- has completed
    k_noalloc_rows<<<grid, 32 * warps_per_cta, 0, stream>>>(bufs->army, bufs->owner, bufs->terrain,
                                                            static_cast<uint32_t *>(scratch), (int)N, (int)P, HW, S, BW);
    if (cudaGetLastError() != cudaSuccess) return GEN_ERR_CUDA;
    gen::env_count_launch(env);
    b.bitboards = static_cast<uint32_t *>(scratch);
    return gen_step(env, &b, d_actions, cuda_stream);
}
