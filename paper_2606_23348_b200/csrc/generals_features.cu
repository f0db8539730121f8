// generals_features.cu -- gen_features: the 38-channel feature tensor of PAPER.md Appendix A and
// Table IV, R35.  One streaming kernel, HBM-write-bound: per game it reads the three state
// planes (4 B per cell), the per-player memory (<= 35 B per cell and player) and writes 38 float planes per player
// (152 B per cell and player).  Nothing here is a contraction; the work per cell is a handful of selects, so the
// design is all about the store stream: one thread owns four consecutive cells of one player's view and issues 38
// 16-byte streaming stores, a warp covers 512 contiguous bytes of each plane; a few CTAs of 288 threads per SM keep
// hundreds of KB of stores in flight per SM, far beyond what the HBM latency-bandwidth product asks for.
//
// Visibility (own cells and their 8 neighbours) is rebuilt from the owner plane, independent of which
// observation format the step kernel was asked for: owner bytes -> one row word per player and row in shared
// memory -> (up | mid | down) dilated by one bit each way.
#include <cuda_runtime.h>
#include <cstdint>

#include "generals_features.h"

namespace gen {

namespace {

constexpr int FEAT_C = 38;
constexpr int FEAT_HIST = 7;
constexpr int FEAT_RING = 8;

__device__ __forceinline__ void st4(float *p, float a, float b, float c, float d) {
    __stcs(reinterpret_cast<float4 *>(p), make_float4(a, b, c, d));
}

__device__ __forceinline__ void unpack4(uint2 v, int (&o)[4]) {  // four int16 in 8 bytes
    o[0] = (int16_t)(v.x & 0xffffu); o[1] = (int16_t)(v.x >> 16);
    o[2] = (int16_t)(v.y & 0xffffu); o[3] = (int16_t)(v.y >> 16);
}

__device__ __forceinline__ uint2 pack4(const int (&v)[4]) {
    return make_uint2((uint32_t)(v[0] & 0xffff) | ((uint32_t)(v[1] & 0xffff) << 16),
                      (uint32_t)(v[2] & 0xffff) | ((uint32_t)(v[3] & 0xffff) << 16));
}

}  // namespace

// grid = ceil(N / G) CTAs; a CTA serves G games with 2 * Q threads each (Q = S / 4 quads per plane).
// dynamic shared memory: [G][S] owner bytes | [G][2][H + 2] own-row words (rows 0 and H + 1 stay zero)
__global__ void __launch_bounds__(512) k_features(const FeatParams fp) {
    extern __shared__ __align__(16) unsigned char smem[];
    const int S = fp.S, Q = S >> 2, H = fp.H, W = fp.W, HW = fp.HW, G = fp.G;
    int8_t *s_owner = reinterpret_cast<int8_t *>(smem);
    uint32_t *s_rows = reinterpret_cast<uint32_t *>(smem + (size_t)G * S);
    const int tid = threadIdx.x, nthr = blockDim.x;
    const int g0 = blockIdx.x * G;
    const int ng = min(G, fp.N - g0);

    // phase 0: owner planes of this CTA's games -> shared memory (16-byte loads; S is a multiple of 16)
    {
        const int4 *src = reinterpret_cast<const int4 *>(fp.owner + (size_t)g0 * S);
        int4 *dst = reinterpret_cast<int4 *>(s_owner);
        for (int i = tid; i < ng * (S >> 4); i += nthr) dst[i] = __ldg(src + i);
        for (int i = tid; i < G * 2 * (H + 2); i += nthr) s_rows[i] = 0u;
    }
    __syncthreads();
    // phase 1: one thread per (game, player, row) packs "owned by p" into a row word
    for (int i = tid; i < ng * 2 * H; i += nthr) {
        const int gl = i / (2 * H), rem = i - gl * 2 * H, p = rem / H, r = rem - p * H;
        const int8_t *row = s_owner + gl * S + r * W;
        uint32_t w = 0;
        for (int c = 0; c < W; ++c) w |= (uint32_t)(row[c] == p) << c;
        s_rows[(gl * 2 + p) * (H + 2) + r + 1] = w;
    }
    __syncthreads();

    // phase 2: one thread per (game, player, quad)
    const int per_game = 2 * Q;
    const int gl = tid / per_game;
    if (gl >= ng) return;
    const int rem = tid - gl * per_game, p = rem / Q, q = rem - p * Q;
    const int g = g0 + gl, opp = 1 - p;
    const size_t gp = (size_t)g * 2 + p;
    const int c0 = 4 * q;

    const int t = __ldg(fp.turn + g);
    const int2 land2 = __ldg(reinterpret_cast<const int2 *>(fp.land) + g);
    const int2 tot2 = __ldg(reinterpret_cast<const int2 *>(fp.army_total) + g);

    int army[4], own[4], terr[4];
    unpack4(__ldg(reinterpret_cast<const uint2 *>(fp.army + (size_t)g * S + c0)), army);
    {
        const uint32_t o4 = *reinterpret_cast<const uint32_t *>(s_owner + gl * S + c0);
        const uint32_t t4 = __ldg(reinterpret_cast<const uint32_t *>(fp.terrain + (size_t)g * S + c0));
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            own[j] = (int8_t)((o4 >> (8 * j)) & 0xffu);
            terr[j] = (int)((t4 >> (8 * j)) & 0xffu);
        }
    }

    // the per-episode memory; a game at turn 0 starts from an empty one (R35), whatever the buffer holds
    uint8_t *mb = fp.mem_bits + gp * S + c0;
    int16_t *la = fp.last_army + gp * S + c0;
    int32_t *ls = fp.last_seen + gp * S + c0;
    int16_t *hist = fp.hist + gp * FEAT_RING * 2 * S + c0;   // [slot][kind][S]
    uint32_t bits4 = 0;
    int last_a[4] = {0, 0, 0, 0};
    int4 seen4 = make_int4(0, 0, 0, 0);                       // turn of the last sighting + 1, 0 = never
    if (t > 0) {
        bits4 = *reinterpret_cast<const uint32_t *>(mb);
        unpack4(*reinterpret_cast<const uint2 *>(la), last_a);
        seen4 = *reinterpret_cast<const int4 *>(ls);
    }
    // frames t-1 .. t-7 of own_army / enemy_army (0 before the episode's first frame)
    uint2 hown[FEAT_HIST], hen[FEAT_HIST];
#pragma unroll
    for (int k = 0; k < FEAT_HIST; ++k) {
        hown[k] = make_uint2(0u, 0u);
        hen[k] = make_uint2(0u, 0u);
        if (t - k - 1 >= 0) {
            const int slot = (t - k - 1) & (FEAT_RING - 1);
            hown[k] = *reinterpret_cast<const uint2 *>(hist + (size_t)(slot * 2 + 0) * S);
            hen[k] = *reinterpret_cast<const uint2 *>(hist + (size_t)(slot * 2 + 1) * S);
        }
    }

    // per-cell quantities
    const uint32_t *rows = s_rows + (gl * 2 + p) * (H + 2);
    int vis[4], valid[4], colv[4], rowv[4], own_a[4], en_a[4], en_vis[4];
    int seen[4] = {seen4.x, seen4.y, seen4.z, seen4.w};
    uint32_t newbits4 = bits4;
    bool any_en = false;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const int c = c0 + j;
        valid[j] = c < HW;
        const int r = valid[j] ? c / W : 0, col = valid[j] ? c - r * W : 0;
        rowv[j] = r; colv[j] = col;
        uint32_t v = rows[r] | rows[r + 1] | rows[r + 2];
        v |= (v << 1) | (v >> 1);
        vis[j] = valid[j] ? (int)((v >> col) & 1u) : 0;
        own_a[j] = (valid[j] && own[j] == p) ? army[j] : 0;
        en_vis[j] = vis[j] && own[j] == opp;
        en_a[j] = en_vis[j] ? army[j] : 0;
        uint32_t b = (uint32_t)vis[j] | ((uint32_t)en_vis[j] << 1);
        if (vis[j]) b |= (terr[j] == 3 ? 4u : 0u) | (terr[j] == 2 ? 8u : 0u) | (terr[j] == 1 ? 16u : 0u);
        newbits4 |= b << (8 * j);
        if (en_vis[j]) { last_a[j] = army[j]; seen[j] = t + 1; any_en = true; }
    }
    // fold into the memory (stores only where something changed)
    if (newbits4 != bits4 || t == 0) *reinterpret_cast<uint32_t *>(mb) = newbits4;
    if (any_en || t == 0) {
        *reinterpret_cast<uint2 *>(la) = pack4(last_a);
        *reinterpret_cast<int4 *>(ls) = make_int4(seen[0], seen[1], seen[2], seen[3]);
    }
    {
        const int slot = t & (FEAT_RING - 1);
        *reinterpret_cast<uint2 *>(hist + (size_t)(slot * 2 + 0) * S) = pack4(own_a);
        *reinterpret_cast<uint2 *>(hist + (size_t)(slot * 2 + 1) * S) = pack4(en_a);
    }

    // Table IV, channel by channel
    float *out = fp.feat + gp * FEAT_C * S + c0;
    float f[4];
#define EMIT(ch, expr)                                                     \
    {                                                                      \
        _Pragma("unroll") for (int j = 0; j < 4; ++j) f[j] = valid[j] ? (float)(expr) : 0.0f; \
        st4(out + (size_t)(ch) * S, f[0], f[1], f[2], f[3]);               \
    }
    EMIT(0, vis[j] ? army[j] : 0)
    EMIT(1, own_a[j])
    EMIT(2, en_a[j])
    EMIT(3, (vis[j] && own[j] == -1) ? army[j] : 0)
#pragma unroll
    for (int k = 0; k < 5; ++k) EMIT(4 + k, (newbits4 >> (8 * j + k)) & 1u)
    EMIT(9, vis[j] && own[j] == -1)
    EMIT(10, own[j] == p)
    EMIT(11, en_vis[j])
    EMIT(12, !vis[j])
    EMIT(13, !vis[j] && ((newbits4 >> (8 * j)) & 0x1cu) != 0u)
    {
        const float ft = (float)t, tick = (float)(t % 50) / 50.0f;
        const float l_me = (float)(p ? land2.y : land2.x), a_me = (float)(p ? tot2.y : tot2.x);
        const float l_op = (float)(p ? land2.x : land2.y), a_op = (float)(p ? tot2.x : tot2.y);
        EMIT(14, ft)
        EMIT(15, tick)
        EMIT(16, l_me)
        EMIT(17, a_me)
        EMIT(18, l_op)
        EMIT(19, a_op)
    }
    EMIT(20, last_a[j])
    EMIT(21, (seen[j] == 0 || en_vis[j]) ? 0.0f : logf(1.0f + (float)(t - (seen[j] - 1))) / 5.0f)
    {
        const float wx = (float)(W - 1), hy = (float)(H - 1);
        EMIT(22, W > 1 ? (float)colv[j] / wx : 0.0f)
        EMIT(23, H > 1 ? (float)rowv[j] / hy : 0.0f)
    }
    // deltas: frame(t-k) - frame(t-k-1), 0 when t-k-1 < 0
    {
        int cur_o[4], cur_e[4], prev[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) { cur_o[j] = own_a[j]; cur_e[j] = en_a[j]; }
#pragma unroll
        for (int k = 0; k < FEAT_HIST; ++k) {
            const bool have = t - k - 1 >= 0;
            unpack4(hown[k], prev);
            EMIT(24 + k, have ? cur_o[j] - prev[j] : 0)
#pragma unroll
            for (int j = 0; j < 4; ++j) cur_o[j] = prev[j];
            unpack4(hen[k], prev);
            EMIT(31 + k, have ? cur_e[j] - prev[j] : 0)
#pragma unroll
            for (int j = 0; j < 4; ++j) cur_e[j] = prev[j];
        }
    }
#undef EMIT
}

cudaError_t launch_features(const FeatParams &fp, cudaStream_t stream) {
    const int per_game = 2 * (fp.S >> 2);
    const int threads = (fp.G * per_game + 31) / 32 * 32;
    const size_t smem = (size_t)fp.G * fp.S + (size_t)fp.G * 2 * (fp.H + 2) * 4;
    const int grid = (fp.N + fp.G - 1) / fp.G;
    k_features<<<grid, threads, smem, stream>>>(fp);
    return cudaGetLastError();
}

}  // namespace gen
