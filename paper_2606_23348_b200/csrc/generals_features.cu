// generals_features.cu -- gen_features: the 38-channel feature tensor of PAPER.md Appendix A and
// Table IV, R35.  One streaming kernel, HBM-write-bound: per game it reads the three state
// planes (4 B per cell), the per-player memory (<= 35 B per cell and player) and writes 38 float planes per player
// (152 B per cell and player).  Nothing here is a contraction; the work per cell is a handful of selects, so the
// design is all about the store stream: one thread owns four consecutive cells of one player's view and issues 38
// 16-byte streaming stores, a warp covers 512 contiguous bytes of each plane, three CTAs of 288 threads per SM
// keep hundreds of KB of stores in flight.  To stay off the issue and conversion pipes the kernel is compiled for
// the paper-sized boards (no integer division, channel offsets as store immediates), army values become floats by
// a byte permute and one add (no I2F), flags by a select, and the two coordinate planes come from a table built
// once per CTA.
//
// Visibility (own cells and their 8 neighbours) is rebuilt from the owner plane, independent of which
// observation format the step kernel was asked for: owner bytes -> one row word per player and row in shared
// memory -> (up | mid | down) dilated by one bit each way.
#include <cuda_bf16.h>
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
// the bfloat16 variant (R37): each fp32 value rounded once, ties to even; four cells = one 8-byte store
__device__ __forceinline__ void st4(__nv_bfloat16 *p, float a, float b, float c, float d) {
    const __nv_bfloat162 lo = __floats2bfloat162_rn(a, b), hi = __floats2bfloat162_rn(c, d);
    __stcs(reinterpret_cast<uint2 *>(p), make_uint2(*reinterpret_cast<const uint32_t *>(&lo),
                                                     *reinterpret_cast<const uint32_t *>(&hi)));
}

// a non-negative int16 (army counts, R21) as a float without a conversion instruction: drop its 16 bits into the
// mantissa of 2^23 and subtract 2^23 (exact)
__device__ __forceinline__ float lo16f(uint32_t v) {
    return __uint_as_float(__byte_perm(v, 0x4B000000u, 0x7610)) - 8388608.0f;
}
__device__ __forceinline__ float hi16f(uint32_t v) {
    return __uint_as_float(__byte_perm(v, 0x4B000000u, 0x7632)) - 8388608.0f;
}
__device__ __forceinline__ void unpack4f(uint2 v, float (&o)[4]) {
    o[0] = lo16f(v.x); o[1] = hi16f(v.x); o[2] = lo16f(v.y); o[3] = hi16f(v.y);
}
__device__ __forceinline__ uint32_t pack2(uint32_t lo, uint32_t hi) { return (lo & 0xffffu) | (hi << 16); }

}  // namespace

// grid = ceil(N / G) CTAs; a CTA serves G games with 2 * Q threads each (Q = S / 4 quads per plane).
// dynamic shared memory: [G][S] owner bytes | [G][2][H + 2] own-row words (rows 0 and H + 1 stay zero) |
// 32 + 32 coordinate floats.  TH, TW: the board this instantiation is compiled for (0 = any board); OUT: float or
// __nv_bfloat16 (R37).
template <int TH, int TW, int MAXT, int MINB, typename OUT>
__global__ void __launch_bounds__(MAXT, MINB) k_features(const FeatParams fp) {
    extern __shared__ __align__(16) unsigned char smem[];
    const int H = TH ? TH : fp.H, W = TW ? TW : fp.W, HW = H * W;
    const int S = TH ? (TH * TW + 15) / 16 * 16 : fp.S, Q = S >> 2, G = fp.G;
    constexpr bool kRowQuads = TW != 0 && TW % 4 == 0;              // a quad never straddles two rows
    constexpr bool kAllValid = TH != 0 && (TH * TW) % 16 == 0;      // no stride padding
    int8_t *s_owner = reinterpret_cast<int8_t *>(smem);
    uint32_t *s_rows = reinterpret_cast<uint32_t *>(smem + (size_t)G * S);
    float *s_cx = reinterpret_cast<float *>(s_rows + G * 2 * (H + 2));
    float *s_cy = s_cx + 32;
    const int tid = threadIdx.x, nthr = blockDim.x;
    const int g0 = blockIdx.x * G;
    const int ng = min(G, fp.N - g0);

    // this thread's (game, player, quad); its global loads are issued before the shared-memory phases
    const int per_game = 2 * Q;
    const int gl = tid / per_game;
    const bool active = gl < ng;
    const int rem = tid - gl * per_game, p = rem / Q, q = rem - p * Q;
    const int g = g0 + gl, opp = 1 - p;
    const size_t gp = (size_t)g * 2 + p;
    const int c0 = 4 * q;

    int t = 0, ph = H, pw = W;                               // playable rows / columns (R36): the rest is a known border
    int2 land2 = make_int2(0, 0), tot2 = make_int2(0, 0);
    uint2 army2 = make_uint2(0u, 0u);
    uint32_t terr4 = 0, bits4 = 0;
    uint2 last2 = make_uint2(0u, 0u);
    int4 seen4 = make_int4(0, 0, 0, 0);                        // turn of the last sighting + 1, 0 = never
    uint2 hown[FEAT_HIST], hen[FEAT_HIST];                     // frames t-1 .. t-7 (0 before the first frame)
    uint8_t *mb = fp.mem_bits + gp * S + c0;
    int16_t *la = fp.last_army + gp * S + c0;
    int32_t *ls = fp.last_seen + gp * S + c0;
    int16_t *hist = fp.hist + gp * FEAT_RING * 2 * S + c0;     // [slot][kind][S]
#pragma unroll
    for (int k = 0; k < FEAT_HIST; ++k) hown[k] = hen[k] = make_uint2(0u, 0u);
    if (active) {
        t = __ldg(fp.turn + g);
        if (fp.play_size) {
            const int v = (int)__ldg(reinterpret_cast<const uint16_t *>(fp.play_size) + g);
            const int vh = (int8_t)(v & 0xff), vw = (int8_t)(v >> 8);
            if (vh > 0) ph = vh;                             // 0 = not recorded (a board written by hand): the full board
            if (vw > 0) pw = vw;
        }
        land2 = __ldg(reinterpret_cast<const int2 *>(fp.land) + g);
        tot2 = __ldg(reinterpret_cast<const int2 *>(fp.army_total) + g);
        army2 = __ldg(reinterpret_cast<const uint2 *>(fp.army + (size_t)g * S + c0));
        terr4 = __ldg(reinterpret_cast<const uint32_t *>(fp.terrain + (size_t)g * S + c0));
        // the per-episode memory; a game at turn 0 starts from an empty one (R35), whatever the buffer holds
        if (t > 0) {
            bits4 = *reinterpret_cast<const uint32_t *>(mb);
            last2 = *reinterpret_cast<const uint2 *>(la);
            seen4 = *reinterpret_cast<const int4 *>(ls);
        }
#pragma unroll
        for (int k = 0; k < FEAT_HIST; ++k) {
            if (t - k - 1 >= 0) {
                const int slot = (t - k - 1) & (FEAT_RING - 1);
                hown[k] = *reinterpret_cast<const uint2 *>(hist + (size_t)(slot * 2 + 0) * S);
                hen[k] = *reinterpret_cast<const uint2 *>(hist + (size_t)(slot * 2 + 1) * S);
            }
        }
    }

    // phase 0: owner planes of this CTA's games -> shared memory (16-byte loads; S is a multiple of 16);
    // coordinate tables col / (W - 1), row / (H - 1) (R35), one IEEE division per entry and CTA
    {
        const int4 *src = reinterpret_cast<const int4 *>(fp.owner + (size_t)g0 * S);
        int4 *dst = reinterpret_cast<int4 *>(s_owner);
        for (int i = tid; i < ng * (S >> 4); i += nthr) dst[i] = __ldg(src + i);
        for (int i = tid; i < G * 2 * (H + 2); i += nthr) s_rows[i] = 0u;
        if (tid < 32) s_cx[tid] = W > 1 ? __fdiv_rn((float)tid, (float)(W - 1)) : 0.0f;
        else if (tid < 64) s_cy[tid - 32] = H > 1 ? __fdiv_rn((float)(tid - 32), (float)(H - 1)) : 0.0f;
    }
    __syncthreads();
    // phase 1: one thread per (game, player, row) packs "owned by p" into a row word
    for (int i = tid; i < ng * 2 * H; i += nthr) {
        const int gi = i / (2 * H), ri = i - gi * 2 * H, pi = ri / H, r = ri - pi * H;
        const int8_t *row = s_owner + gi * S + r * W;
        uint32_t w = 0;
        if (kRowQuads) {          // four cells per word: byte-wise compare, then gather the four flags
#pragma unroll
            for (int c4 = 0; c4 < TW / 4; ++c4) {
                const uint32_t x = reinterpret_cast<const uint32_t *>(row)[c4];
                const uint32_t m = __vcmpeq4(x, pi ? 0x01010101u : 0u) & 0x01010101u;
                w |= ((m * 0x01020408u) >> 24) << (4 * c4);
            }
        } else {
            for (int c = 0; c < W; ++c) w |= (uint32_t)(row[c] == pi) << c;
        }
        s_rows[(gi * 2 + pi) * (H + 2) + r + 1] = w;
    }
    __syncthreads();
    if (!active) return;

    // phase 2: per-cell quantities of the quad
    const uint32_t own4 = *reinterpret_cast<const uint32_t *>(s_owner + gl * S + c0);
    const uint32_t *rows = s_rows + (gl * 2 + p) * (H + 2);
    bool valid[4], vis[4], mine[4], en[4], neu[4];
    int rowj[4], colj[4];
    if (kRowQuads) {
        const bool ok = kAllValid || c0 < HW;
        const int r = ok ? c0 / W : 0, col0 = ok ? c0 - r * W : 0;
        uint32_t v = rows[r] | rows[r + 1] | rows[r + 2];
        v |= (v << 1) | (v >> 1);
        v = ok ? v >> col0 : 0u;
#pragma unroll
        for (int j = 0; j < 4; ++j) { valid[j] = ok; vis[j] = (v >> j) & 1u; rowj[j] = r; colj[j] = col0 + j; }
    } else {
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int c = c0 + j;
            valid[j] = c < HW;
            const int r = valid[j] ? c / W : 0, col = valid[j] ? c - r * W : 0;
            uint32_t v = rows[r] | rows[r + 1] | rows[r + 2];
            v |= (v << 1) | (v >> 1);
            vis[j] = valid[j] && ((v >> col) & 1u);
            rowj[j] = r; colj[j] = col;
        }
    }
    const uint32_t a16[4] = {army2.x & 0xffffu, army2.x >> 16, army2.y & 0xffffu, army2.y >> 16};
    uint32_t l16[4] = {last2.x & 0xffffu, last2.x >> 16, last2.y & 0xffffu, last2.y >> 16};
    int seen[4] = {seen4.x, seen4.y, seen4.z, seen4.w};
    uint32_t own_f[4], en_f[4];                                  // this turn's history frames
    uint32_t newbits4 = bits4;
    bool any_en = false;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const int o = (int8_t)((own4 >> (8 * j)) & 0xffu);
        const uint32_t tr = (terr4 >> (8 * j)) & 0xffu;
        mine[j] = valid[j] && o == p;
        en[j] = vis[j] && o == opp;
        neu[j] = vis[j] && o == -1;
        uint32_t b = (uint32_t)vis[j] | ((uint32_t)en[j] << 1);
        if (vis[j]) b |= (tr == 3u ? 4u : 0u) | (tr == 2u ? 8u : 0u) | (tr == 1u ? 16u : 0u);
        if (valid[j] && (rowj[j] >= ph || colj[j] >= pw)) b |= 16u;   // Table IV ch 8: "U known padded border"
        newbits4 |= b << (8 * j);
        if (en[j]) { l16[j] = a16[j]; seen[j] = t + 1; any_en = true; }
        own_f[j] = mine[j] ? a16[j] : 0u;
        en_f[j] = en[j] ? a16[j] : 0u;
    }
    const uint2 newlast2 = make_uint2(pack2(l16[0], l16[1]), pack2(l16[2], l16[3]));
    // fold into the memory (stores only where something changed)
    if (newbits4 != bits4 || t == 0) *reinterpret_cast<uint32_t *>(mb) = newbits4;
    if (any_en || t == 0) {
        *reinterpret_cast<uint2 *>(la) = newlast2;
        *reinterpret_cast<int4 *>(ls) = make_int4(seen[0], seen[1], seen[2], seen[3]);
    }
    {
        const int slot = t & (FEAT_RING - 1);
        *reinterpret_cast<uint2 *>(hist + (size_t)(slot * 2 + 0) * S) =
            make_uint2(pack2(own_f[0], own_f[1]), pack2(own_f[2], own_f[3]));
        *reinterpret_cast<uint2 *>(hist + (size_t)(slot * 2 + 1) * S) =
            make_uint2(pack2(en_f[0], en_f[1]), pack2(en_f[2], en_f[3]));
    }

    // Table IV, channel by channel.  EMIT(ch, expr): expr is a float in terms of j; padding cells are 0.
    OUT *out = reinterpret_cast<OUT *>(fp.feat) + gp * FEAT_C * S + c0;
    float f[4], fa[4];
    unpack4f(army2, fa);
#define EMIT(ch, expr)                                                                                  \
    {                                                                                                   \
        _Pragma("unroll") for (int j = 0; j < 4; ++j) f[j] = (kAllValid || valid[j]) ? (expr) : 0.0f;  \
        st4(out + (size_t)(ch) * S, f[0], f[1], f[2], f[3]);                                            \
    }
    // deltas first (the 28 registers of history frames retire early): frame(t-k) - frame(t-k-1), 0 when t-k-1 < 0;
    // frames are exact small integers in fp32, so the float difference is exact
    {
        float cur_o[4], cur_e[4], prev[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) { cur_o[j] = mine[j] ? fa[j] : 0.0f; cur_e[j] = en[j] ? fa[j] : 0.0f; }
#pragma unroll
        for (int k = 0; k < FEAT_HIST; ++k) {
            const bool have = t - k - 1 >= 0;
            unpack4f(hown[k], prev);
            EMIT(24 + k, have ? cur_o[j] - prev[j] : 0.0f)
#pragma unroll
            for (int j = 0; j < 4; ++j) cur_o[j] = prev[j];
            unpack4f(hen[k], prev);
            EMIT(31 + k, have ? cur_e[j] - prev[j] : 0.0f)
#pragma unroll
            for (int j = 0; j < 4; ++j) cur_e[j] = prev[j];
        }
    }
    EMIT(0, vis[j] ? fa[j] : 0.0f)
    EMIT(1, mine[j] ? fa[j] : 0.0f)
    EMIT(2, en[j] ? fa[j] : 0.0f)
    EMIT(3, neu[j] ? fa[j] : 0.0f)
#pragma unroll
    for (int k = 0; k < 5; ++k) EMIT(4 + k, ((newbits4 >> (8 * j + k)) & 1u) ? 1.0f : 0.0f)
    EMIT(9, neu[j] ? 1.0f : 0.0f)
    EMIT(10, mine[j] ? 1.0f : 0.0f)
    EMIT(11, en[j] ? 1.0f : 0.0f)
    EMIT(12, vis[j] ? 0.0f : 1.0f)
    EMIT(13, (!vis[j] && ((newbits4 >> (8 * j)) & 0x1cu) != 0u) ? 1.0f : 0.0f)
    {
        const float ft = (float)t, tick = __fdiv_rn((float)(t % 50), 50.0f);
        const float l_me = (float)(p ? land2.y : land2.x), a_me = (float)(p ? tot2.y : tot2.x);
        const float l_op = (float)(p ? land2.x : land2.y), a_op = (float)(p ? tot2.x : tot2.y);
        EMIT(14, ft)
        EMIT(15, tick)
        EMIT(16, l_me)
        EMIT(17, a_me)
        EMIT(18, l_op)
        EMIT(19, a_op)
    }
    {
        float fl[4], age[4] = {0.0f, 0.0f, 0.0f, 0.0f};
        unpack4f(newlast2, fl);
        EMIT(20, fl[j])
        // log(1 + turns since the last sighting) / 5; 0 where the enemy was never seen or is visible now (R35).
        // Most quads have no remembered enemy cell: the transcendental path is skipped for them.
        bool need = false;
#pragma unroll
        for (int j = 0; j < 4; ++j) need |= seen[j] != 0 && !en[j];
        if (need) {
#pragma unroll
            for (int j = 0; j < 4; ++j)
                if (seen[j] != 0 && !en[j]) age[j] = __fdiv_rn(logf(1.0f + (float)(t - (seen[j] - 1))), 5.0f);
        }
        EMIT(21, age[j])
    }
    EMIT(22, s_cx[colj[j]])
    EMIT(23, s_cy[rowj[j]])
#undef EMIT
}

// ------------------------------------------------------------------------------------------------
// More than two players (R38; the same observation interface in 1v1, 2v2 and free-for-all), any board.  "The
// opponent" is every player off the agent's team, visibility is the team's, the opponent's scoreboard entries are
// sums over the enemies.  One CTA per game; its threads loop over the P * Q (player, quad) items.  The per-item work
// is the 1v1 kernel's (kept apart so that the tuned 1v1 path stays exactly what it is); the team test replaces the
// "owner == 1 - p" compare.  dynamic shared memory: [S] owner bytes | [teams][H + 2] row words of the team's cells |
// 32 + 32 coordinate floats | 8 + 8 scoreboard ints.
template <typename OUT>
__global__ void __launch_bounds__(256, 2) k_features_mp(const FeatParams fp) {
    extern __shared__ __align__(16) unsigned char smem[];
    const int S = fp.S, Q = S >> 2, H = fp.H, W = fp.W, HW = fp.HW, P = fp.P, ts = fp.team_size;
    const int NT = (P + ts - 1) / ts;
    int8_t *s_owner = reinterpret_cast<int8_t *>(smem);
    uint32_t *s_rows = reinterpret_cast<uint32_t *>(smem + S);
    float *s_cx = reinterpret_cast<float *>(s_rows + NT * (H + 2));
    float *s_cy = s_cx + 32;
    int *s_land = reinterpret_cast<int *>(s_cy + 32), *s_tot = s_land + 8;
    const int tid = threadIdx.x, nthr = blockDim.x;
    const int g = blockIdx.x;
    {
        const int4 *src = reinterpret_cast<const int4 *>(fp.owner + (size_t)g * S);
        int4 *dst = reinterpret_cast<int4 *>(s_owner);
        for (int i = tid; i < (S >> 4); i += nthr) dst[i] = __ldg(src + i);
        for (int i = tid; i < NT * (H + 2); i += nthr) s_rows[i] = 0u;
        if (tid < 32) s_cx[tid] = W > 1 ? __fdiv_rn((float)tid, (float)(W - 1)) : 0.0f;
        else if (tid < 64) s_cy[tid - 32] = H > 1 ? __fdiv_rn((float)(tid - 32), (float)(H - 1)) : 0.0f;
        else if (tid < 64 + P) {
            s_land[tid - 64] = __ldg(fp.land + (size_t)g * P + (tid - 64));
            s_tot[tid - 64] = __ldg(fp.army_total + (size_t)g * P + (tid - 64));
        }
    }
    __syncthreads();
    for (int i = tid; i < NT * H; i += nthr) {      // one thread per (team, row): the cells of the team's members
        const int T = i / H, r = i - T * H;
        const int8_t *row = s_owner + r * W;
        uint32_t w = 0;
        for (int c = 0; c < W; ++c) {
            const int o = row[c];
            w |= (uint32_t)(o >= 0 && o / ts == T) << c;
        }
        s_rows[T * (H + 2) + r + 1] = w;
    }
    __syncthreads();

    const int t = __ldg(fp.turn + g);
    int ph = H, pw = W;
    if (fp.play_size) {
        const int v = (int)__ldg(reinterpret_cast<const uint16_t *>(fp.play_size) + g);
        const int vh = (int8_t)(v & 0xff), vw = (int8_t)(v >> 8);
        if (vh > 0) ph = vh;
        if (vw > 0) pw = vw;
    }
    for (int item = tid; item < P * Q; item += nthr) {
        const int p = item / Q, q = item - p * Q, team = p / ts, c0 = 4 * q;
        const size_t gp = (size_t)g * P + p;
        const uint2 army2 = __ldg(reinterpret_cast<const uint2 *>(fp.army + (size_t)g * S + c0));
        const uint32_t terr4 = __ldg(reinterpret_cast<const uint32_t *>(fp.terrain + (size_t)g * S + c0));
        const uint32_t own4 = *reinterpret_cast<const uint32_t *>(s_owner + c0);
        uint8_t *mb = fp.mem_bits + gp * S + c0;
        int16_t *la = fp.last_army + gp * S + c0;
        int32_t *ls = fp.last_seen + gp * S + c0;
        int16_t *hist = fp.hist + gp * FEAT_RING * 2 * S + c0;
        uint32_t bits4 = 0;
        uint2 last2 = make_uint2(0u, 0u);
        int4 seen4 = make_int4(0, 0, 0, 0);
        if (t > 0) {
            bits4 = *reinterpret_cast<const uint32_t *>(mb);
            last2 = *reinterpret_cast<const uint2 *>(la);
            seen4 = *reinterpret_cast<const int4 *>(ls);
        }
        uint2 hown[FEAT_HIST], hen[FEAT_HIST];
#pragma unroll
        for (int k = 0; k < FEAT_HIST; ++k) {
            hown[k] = hen[k] = make_uint2(0u, 0u);
            if (t - k - 1 >= 0) {
                const int slot = (t - k - 1) & (FEAT_RING - 1);
                hown[k] = *reinterpret_cast<const uint2 *>(hist + (size_t)(slot * 2 + 0) * S);
                hen[k] = *reinterpret_cast<const uint2 *>(hist + (size_t)(slot * 2 + 1) * S);
            }
        }
        int l_op_i = 0, a_op_i = 0;
        for (int e = 0; e < P; ++e)
            if (e / ts != team) { l_op_i += s_land[e]; a_op_i += s_tot[e]; }

        const uint32_t *rows = s_rows + team * (H + 2);
        bool valid[4], vis[4], mine[4], en[4], neu[4];
        int rowj[4], colj[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int c = c0 + j;
            valid[j] = c < HW;
            const int r = valid[j] ? c / W : 0, col = valid[j] ? c - r * W : 0;
            uint32_t v = rows[r] | rows[r + 1] | rows[r + 2];
            v |= (v << 1) | (v >> 1);
            vis[j] = valid[j] && ((v >> col) & 1u);
            rowj[j] = r; colj[j] = col;
        }
        const uint32_t a16[4] = {army2.x & 0xffffu, army2.x >> 16, army2.y & 0xffffu, army2.y >> 16};
        uint32_t l16[4] = {last2.x & 0xffffu, last2.x >> 16, last2.y & 0xffffu, last2.y >> 16};
        int seen[4] = {seen4.x, seen4.y, seen4.z, seen4.w};
        uint32_t own_f[4], en_f[4];
        uint32_t newbits4 = bits4;
        bool any_en = false;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int o = (int8_t)((own4 >> (8 * j)) & 0xffu);
            const uint32_t tr = (terr4 >> (8 * j)) & 0xffu;
            mine[j] = valid[j] && o == p;
            en[j] = vis[j] && o >= 0 && o / ts != team;
            neu[j] = vis[j] && o == -1;
            uint32_t b = (uint32_t)vis[j] | ((uint32_t)en[j] << 1);
            if (vis[j]) b |= (tr == 3u ? 4u : 0u) | (tr == 2u ? 8u : 0u) | (tr == 1u ? 16u : 0u);
            if (valid[j] && (rowj[j] >= ph || colj[j] >= pw)) b |= 16u;
            newbits4 |= b << (8 * j);
            if (en[j]) { l16[j] = a16[j]; seen[j] = t + 1; any_en = true; }
            own_f[j] = mine[j] ? a16[j] : 0u;
            en_f[j] = en[j] ? a16[j] : 0u;
        }
        const uint2 newlast2 = make_uint2(pack2(l16[0], l16[1]), pack2(l16[2], l16[3]));
        if (newbits4 != bits4 || t == 0) *reinterpret_cast<uint32_t *>(mb) = newbits4;
        if (any_en || t == 0) {
            *reinterpret_cast<uint2 *>(la) = newlast2;
            *reinterpret_cast<int4 *>(ls) = make_int4(seen[0], seen[1], seen[2], seen[3]);
        }
        {
            const int slot = t & (FEAT_RING - 1);
            *reinterpret_cast<uint2 *>(hist + (size_t)(slot * 2 + 0) * S) =
                make_uint2(pack2(own_f[0], own_f[1]), pack2(own_f[2], own_f[3]));
            *reinterpret_cast<uint2 *>(hist + (size_t)(slot * 2 + 1) * S) =
                make_uint2(pack2(en_f[0], en_f[1]), pack2(en_f[2], en_f[3]));
        }

        OUT *out = reinterpret_cast<OUT *>(fp.feat) + gp * FEAT_C * S + c0;
        float f[4], fa[4];
        unpack4f(army2, fa);
#define EMIT(ch, expr)                                                                     \
    {                                                                                      \
        _Pragma("unroll") for (int j = 0; j < 4; ++j) f[j] = valid[j] ? (expr) : 0.0f;    \
        st4(out + (size_t)(ch) * S, f[0], f[1], f[2], f[3]);                               \
    }
        {
            float cur_o[4], cur_e[4], prev[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) { cur_o[j] = mine[j] ? fa[j] : 0.0f; cur_e[j] = en[j] ? fa[j] : 0.0f; }
#pragma unroll
            for (int k = 0; k < FEAT_HIST; ++k) {
                const bool have = t - k - 1 >= 0;
                unpack4f(hown[k], prev);
                EMIT(24 + k, have ? cur_o[j] - prev[j] : 0.0f)
#pragma unroll
                for (int j = 0; j < 4; ++j) cur_o[j] = prev[j];
                unpack4f(hen[k], prev);
                EMIT(31 + k, have ? cur_e[j] - prev[j] : 0.0f)
#pragma unroll
                for (int j = 0; j < 4; ++j) cur_e[j] = prev[j];
            }
        }
        EMIT(0, vis[j] ? fa[j] : 0.0f)
        EMIT(1, mine[j] ? fa[j] : 0.0f)
        EMIT(2, en[j] ? fa[j] : 0.0f)
        EMIT(3, neu[j] ? fa[j] : 0.0f)
#pragma unroll
        for (int k = 0; k < 5; ++k) EMIT(4 + k, ((newbits4 >> (8 * j + k)) & 1u) ? 1.0f : 0.0f)
        EMIT(9, neu[j] ? 1.0f : 0.0f)
        EMIT(10, mine[j] ? 1.0f : 0.0f)
        EMIT(11, en[j] ? 1.0f : 0.0f)
        EMIT(12, vis[j] ? 0.0f : 1.0f)
        EMIT(13, (!vis[j] && ((newbits4 >> (8 * j)) & 0x1cu) != 0u) ? 1.0f : 0.0f)
        {
            const float ft = (float)t, tick = __fdiv_rn((float)(t % 50), 50.0f);
            const float l_me = (float)s_land[p], a_me = (float)s_tot[p];
            const float l_op = (float)l_op_i, a_op = (float)a_op_i;
            EMIT(14, ft)
            EMIT(15, tick)
            EMIT(16, l_me)
            EMIT(17, a_me)
            EMIT(18, l_op)
            EMIT(19, a_op)
        }
        {
            float fl[4], age[4] = {0.0f, 0.0f, 0.0f, 0.0f};
            unpack4f(newlast2, fl);
            EMIT(20, fl[j])
#pragma unroll
            for (int j = 0; j < 4; ++j)
                if (seen[j] != 0 && !en[j]) age[j] = __fdiv_rn(logf(1.0f + (float)(t - (seen[j] - 1))), 5.0f);
            EMIT(21, age[j])
        }
        EMIT(22, s_cx[colj[j]])
        EMIT(23, s_cy[rowj[j]])
#undef EMIT
    }
}

namespace {

template <int TH, int TW, int MAXT, int MINB>
cudaError_t launch_one(const FeatParams &fp, int threads, cudaStream_t stream) {
    const size_t smem = (size_t)fp.G * fp.S + (size_t)fp.G * 2 * (fp.H + 2) * 4 + 64 * 4;
    const int grid = (fp.N + fp.G - 1) / fp.G;
    if (fp.bf16) k_features<TH, TW, MAXT, MINB, __nv_bfloat16><<<grid, threads, smem, stream>>>(fp);
    else k_features<TH, TW, MAXT, MINB, float><<<grid, threads, smem, stream>>>(fp);
    return cudaGetLastError();
}

}  // namespace

// Board-specialised instantiations for the paper-sized 1v1 boards (BASELINE configs 1 and 2-4, the paper's own 23x23),
// else the generic one.
// ================================================================================================
// The two temporal tokens' windows (reading R39): for game g and agent p, win[g][p][0][i] /
// win[g][p][1][i] = the enemies' summed army total / land count at turn t - 511 + i of the current episode (t = turn[g];
// i = 511 is now), 0 before the episode's first turn.  The source is the scoreboard ring of R34, slot (turn mod 512) =
// (land[q], army[q]) of every player q.  One CTA of 512 threads per game, thread i owns window entry i: the slots it
// reads are consecutive in i (one wrap), so the loads are 2P * 4-byte runs side by side and every store instruction
// covers 2 KB of one window.  HBM-bound: 4 KB * P read, 4 KB * P written per game.
template <int NP>
__global__ void __launch_bounds__(512) k_history_windows(const int32_t *__restrict__ ring, const int32_t *__restrict__ turn,
                                                         int32_t *__restrict__ win, int P, int team_size) {
    const int g = blockIdx.x, i = threadIdx.x;
    const int t = __ldg(turn + g);
    const int tt = t - 511 + i;
    int32_t v[2 * NP];
#pragma unroll
    for (int k = 0; k < 2 * NP; ++k) v[k] = 0;
    if (tt >= 0) {
        const int32_t *slot = ring + ((size_t)g * 512 + (size_t)(tt & 511)) * 2 * P;
        if (NP == 2) {
            const int4 q = __ldcs(reinterpret_cast<const int4 *>(slot));   // 2P ints = 16 bytes at P = 2
            v[0] = q.x; v[1] = q.y; v[2] = q.z; v[3] = q.w;
        } else {
#pragma unroll
            for (int k = 0; k < NP; ++k)
                if (k < P) {
                    const int2 q = __ldcs(reinterpret_cast<const int2 *>(slot) + k);
                    v[2 * k] = q.x; v[2 * k + 1] = q.y;
                }
        }
    }
    int32_t land_all = 0, army_all = 0;
#pragma unroll
    for (int k = 0; k < NP; ++k) { land_all += v[2 * k]; army_all += v[2 * k + 1]; }
#pragma unroll
    for (int p = 0; p < NP; ++p) {
        if (p >= P) break;
        int32_t land = land_all, army = army_all;   // everybody, minus the agent's own team
#pragma unroll
        for (int q = 0; q < NP; ++q)
            if (q < P && q / team_size == p / team_size) { land -= v[2 * q]; army -= v[2 * q + 1]; }
        int32_t *out = win + (((size_t)g * P + p) * 2) * 512 + i;
        __stcs(out, army);
        __stcs(out + 512, land);
    }
}

cudaError_t launch_history_windows(const int32_t *ring, const int32_t *turn, int32_t *win, int N, int P, int team_size,
                                   cudaStream_t stream) {
    if (P == 2) k_history_windows<2><<<N, 512, 0, stream>>>(ring, turn, win, P, team_size);
    else if (P <= 4) k_history_windows<4><<<N, 512, 0, stream>>>(ring, turn, win, P, team_size);
    else k_history_windows<8><<<N, 512, 0, stream>>>(ring, turn, win, P, team_size);
    return cudaGetLastError();
}

cudaError_t launch_features(const FeatParams &fp, cudaStream_t stream) {
    if (fp.P != 2 || fp.team_size != 1) {          // R38: the multi-player kernel, one CTA per game
        const int NT = (fp.P + fp.team_size - 1) / fp.team_size;
        const size_t smem = (size_t)fp.S + (size_t)NT * (fp.H + 2) * 4 + 64 * 4 + 16 * 4;
        if (fp.bf16) k_features_mp<__nv_bfloat16><<<fp.N, 256, smem, stream>>>(fp);
        else k_features_mp<float><<<fp.N, 256, smem, stream>>>(fp);
        return cudaGetLastError();
    }
    const int per_game = 2 * (fp.S >> 2);
    const int threads = (fp.G * per_game + 31) / 32 * 32;
    if (threads < 64) return cudaErrorInvalidConfiguration;   // the coordinate tables need two warps
    if (!fp.force_generic && fp.H == 24 && fp.W == 24 && threads <= 288) return launch_one<24, 24, 288, 3>(fp, threads, stream);
    if (!fp.force_generic && fp.H == 23 && fp.W == 23 && threads <= 288) return launch_one<23, 23, 288, 3>(fp, threads, stream);
    if (!fp.force_generic && fp.H == 8 && fp.W == 8 && threads <= 256) return launch_one<8, 8, 256, 4>(fp, threads, stream);
    return launch_one<0, 0, 512, 2>(fp, threads, stream);
}

}  // namespace gen
