// generals_kernels.cuh -- device code of the batched Generals.io step for sm_100a.
//
// One warp owns one game.  The board (int16 army, int8 owner, int8 terrain planes) is staged in
// shared memory; ownership / terrain / "army >= 2" live as FLAT BITBOARDS, one 32-bit word per lane
// (lane j holds cells 32j .. 32j+31), so that fog-of-war dilation, valid-move enumeration and the
// scoreboard are a handful of funnel shifts, shuffles, popcounts and REDUX per game instead of a
// pass over cells.  Per-cell work (mask building, observation planes, digest) runs on 8-cell chunks
// with SIMD-in-register byte arithmetic and 16/8-byte shared and global accesses.
//
// Rules: PAPER.md section IV, readings R1..R32 of DESIGN.md.  This file shares nothing
// with oracle/ (the CPU checker); it is written from the same rules text.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "generals.h"

namespace gen {

constexpr uint32_t FULL = 0xffffffffu;
constexpr int MASK_STRIDE = 128;  // bytes per bitboard staging row (32 words)

enum : uint32_t {
    F_RESET = 1u << 0,         // generate every board first (gen_reset)
    F_SAMPLER = 1u << 1,       // draw actions with the built-in sampler
    F_OBS_PLANES = 1u << 2,    // write observation planes
    F_OBS_EVERY = 1u << 3,     // ... for every step, slot k
    F_DIGEST = 1u << 4,        // chain the observation digest
    F_OBSERVE_ONLY = 1u << 5,  // gen_observe: recount + planes, no turn
    F_SAMPLE_ONLY = 1u << 6,   // gen_sample: actions only
    F_KEEP_EPISODE = 1u << 7,
};

enum : int { T_PLAIN = 0, T_MOUNTAIN = 1, T_CITY = 2, T_GENERAL = 3, T_FOG = 4 };

struct KParams {
    int32_t N, H, W, P, HW, S, NW, NC8;
    int32_t team_size, n_teams;
    int32_t n_cities, city_lo, city_span;
    int32_t dmin, dmax, spawn_exact, max_turns, auto_reset;
    uint32_t rule_flags, gid_base, mountain_thr, key0, key1;
    uint32_t pass_thr, half_thr, bias_thr;
    uint32_t global_step0, flags, recipW;
    int32_t K;
    uint32_t per_warp_bytes, key_bytes;
    gen_buffers b;
    const int32_t *actions;
    int32_t *sample_out;
    uint32_t notcol0[32], notcolL[32], inb[32];
};

// ------------------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon et al., SC'11).  Counter layout of the stream table in DESIGN.md (R24, R30):
// (c0, global game id, c2, domain << 24 | player), key = seed.
enum : uint32_t { DOM_SPAWN = 1, DOM_MOUNTAIN = 2, DOM_CITY = 3, DOM_ACTION = 4 };

__device__ __forceinline__ void philox(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0,
                                       uint32_t k1, uint32_t (&w)[4]) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t h0 = __umulhi(0xD2511F53u, c0), l0 = 0xD2511F53u * c0;
        const uint32_t h1 = __umulhi(0xCD9E8D57u, c2), l1 = 0xCD9E8D57u * c2;
        c0 = h1 ^ c1 ^ k0;
        c2 = h0 ^ c3 ^ k1;
        c1 = l1;
        c3 = l0;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    w[0] = c0; w[1] = c1; w[2] = c2; w[3] = c3;
}

__device__ __forceinline__ uint64_t mix64(uint64_t z) {  // splitmix64 finaliser
    z ^= z >> 30; z *= 0xBF58476D1CE4E5B9ull;
    z ^= z >> 27; z *= 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

// ------------------------------------------------------------------------------------------------
// flat bitboard helpers: lane j holds word j
__device__ __forceinline__ uint32_t bb_shl(uint32_t x, int k, uint32_t lane) {  // bit c -> c + k, 1 <= k <= 32
    uint32_t lo = __shfl_up_sync(FULL, x, 1);
    if (lane == 0) lo = 0;
    return __funnelshift_lc(lo, x, k);
}
__device__ __forceinline__ uint32_t bb_shr(uint32_t x, int k, uint32_t lane) {  // bit c -> c - k
    uint32_t hi = __shfl_down_sync(FULL, x, 1);
    if (lane == 31) hi = 0;
    return __funnelshift_rc(x, hi, k);
}
__device__ __forceinline__ int nth_bit(uint32_t w, uint32_t r) {  // position of the r-th (0-based) set bit
    int pos = 0;
#pragma unroll
    for (int s = 16; s >= 1; s >>= 1) {
        const uint32_t c = __popc((w >> pos) & ((1u << s) - 1u));
        if (r >= c) { r -= c; pos += s; }
    }
    return pos;
}
// cell index of the k-th set bit (0-based, row-major order) of a bitboard; needs k < total popcount
__device__ __forceinline__ int select_kth(uint32_t word, uint32_t k, uint32_t lane) {
    const uint32_t cnt = __popc(word);
    uint32_t incl = cnt;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t v = __shfl_up_sync(FULL, incl, o);
        if (lane >= (uint32_t)o) incl += v;
    }
    const uint32_t b = __ballot_sync(FULL, k < incl);
    const int j = __ffs(b) - 1;
    const uint32_t excl_j = __shfl_sync(FULL, incl - cnt, j);
    const uint32_t wj = __shfl_sync(FULL, word, j);
    return j * 32 + nth_bit(wj, k - excl_j);
}
__device__ __forceinline__ uint32_t mulhi32(uint32_t u, uint32_t n) { return __umulhi(u, n); }

// SIMD-in-register byte helpers
__device__ __forceinline__ uint32_t nib_to_bytes(uint32_t nib) {  // 4 bits -> 4 bytes 0x00 / 0xFF
    return ((nib * 0x00204081u) & 0x01010101u) * 0xFFu;
}
__device__ __forceinline__ uint32_t flags_to_nib(uint32_t f) {  // bit 0 of each byte -> 4 bits
    return (f * 0x01020408u) >> 24;
}
__device__ __forceinline__ uint32_t eq_bytes(uint32_t w, uint32_t pat) {  // 0x01 where byte == pat byte
    const uint32_t x = w ^ pat;
    const uint32_t y = ((x & 0x7F7F7F7Fu) + 0x7F7F7F7Fu) | x;
    return (~y >> 7) & 0x01010101u;
}

template <int NP>
__device__ __forceinline__ uint32_t sel(const uint32_t (&a)[NP], int i) {
    uint32_t v = 0;
#pragma unroll
    for (int q = 0; q < NP; ++q) v = (q == i) ? a[q] : v;
    return v;
}

// ================================================================================================
template <int NP, int WPC>
__global__ void __launch_bounds__(WPC * 32) k_generals(const __grid_constant__ KParams kp) {
    extern __shared__ __align__(16) unsigned char smem[];
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const int H = kp.H, W = kp.W, P = kp.P, HW = kp.HW, S = kp.S, NW = kp.NW, NC8 = kp.NC8;
    const uint32_t flags = kp.flags;
    const gen_buffers &B = kp.b;

    // digest keys (R28): key(c) = mix64((c + 1) * golden gamma) | 1, one table per CTA
    uint64_t *s_key = reinterpret_cast<uint64_t *>(smem);
    if (flags & F_DIGEST) {
        for (int c = threadIdx.x; c < S; c += WPC * 32)
            s_key[c] = (c < HW) ? (mix64((uint64_t)(c + 1) * 0x9E3779B97F4A7C15ull) | 1ull) : 0ull;
        __syncthreads();
    }
    const int g = blockIdx.x * WPC + (int)warp;
    if (g >= kp.N) return;
    const uint32_t gid = kp.gid_base + (uint32_t)g;

    unsigned char *wb = smem + kp.key_bytes + warp * kp.per_warp_bytes;
    int16_t *s_army = reinterpret_cast<int16_t *>(wb);
    int8_t *s_owner = reinterpret_cast<int8_t *>(wb + 2 * S);
    int8_t *s_terr = reinterpret_cast<int8_t *>(wb + 3 * S);
    unsigned char *s_mask = wb + 4 * S;  // (NP + 3) rows of MASK_STRIDE bytes; rows 0..NP-1 double as vis

    const uint32_t notcol0 = kp.notcol0[lane], notcolL = kp.notcolL[lane], inb = kp.inb[lane];
    const uint32_t allp = (1u << P) - 1u;

    // ---- per-game registers (uniform across the warp unless noted) ----
    int turn = 0, winner = -1;
    uint32_t alive = allp, done = 0, episode = 0;
    int tot[NP];                      // army_total, kept incrementally
    uint32_t own[NP], mtn, strct, a2;  // per-lane bitboard words
    bool terrain_dirty = false;
    uint64_t digest = 0;
#pragma unroll
    for (int p = 0; p < NP; ++p) { tot[p] = 0; own[p] = 0; }

    auto team_mask = [&](int p) -> uint32_t {
        const int t = p / kp.team_size;
        return (((1u << kp.team_size) - 1u) << (t * kp.team_size)) & allp;
    };

    // ---------------------------------------------------------------- bitboards from the planes
    auto build_masks = [&]() {
        __syncwarp();
        for (int ch = lane; ch < NC8; ch += 32) {
            const uint2 o = *reinterpret_cast<const uint2 *>(s_owner + 8 * ch);
            const uint2 t = *reinterpret_cast<const uint2 *>(s_terr + 8 * ch);
            const uint4 a = *reinterpret_cast<const uint4 *>(s_army + 8 * ch);
#pragma unroll
            for (int p = 0; p < NP; ++p)
                if (p < P) {
                    const uint32_t pat = 0x01010101u * (uint32_t)p;
                    s_mask[p * MASK_STRIDE + ch] =
                        (unsigned char)(flags_to_nib(eq_bytes(o.x, pat)) | (flags_to_nib(eq_bytes(o.y, pat)) << 4));
                }
            // terrain in {0,1,2,3}: mountain = 01, structure (city / general) = 1x
            const uint32_t sx = (t.x >> 1) & 0x01010101u, sy = (t.y >> 1) & 0x01010101u;
            const uint32_t mx = t.x & ~(t.x >> 1) & 0x01010101u, my = t.y & ~(t.y >> 1) & 0x01010101u;
            s_mask[NP * MASK_STRIDE + ch] = (unsigned char)(flags_to_nib(mx) | (flags_to_nib(my) << 4));
            s_mask[(NP + 1) * MASK_STRIDE + ch] = (unsigned char)(flags_to_nib(sx) | (flags_to_nib(sy) << 4));
            // army >= 2  <=>  (a & 0x7FFE) != 0 for a in [0, 32767]
            const uint32_t y0 = (a.x & 0x7FFE7FFEu) + 0x7FFE7FFEu, y1 = (a.y & 0x7FFE7FFEu) + 0x7FFE7FFEu;
            const uint32_t y2 = (a.z & 0x7FFE7FFEu) + 0x7FFE7FFEu, y3 = (a.w & 0x7FFE7FFEu) + 0x7FFE7FFEu;
            const uint32_t u = (__byte_perm(y0, y1, 0x7531) >> 7) & 0x01010101u;
            const uint32_t v = (__byte_perm(y2, y3, 0x7531) >> 7) & 0x01010101u;
            s_mask[(NP + 2) * MASK_STRIDE + ch] = (unsigned char)(flags_to_nib(u) | (flags_to_nib(v) << 4));
        }
        __syncwarp();
        const bool act = (int)lane < NW;
#pragma unroll
        for (int p = 0; p < NP; ++p)
            own[p] = (act && p < P) ? (reinterpret_cast<const uint32_t *>(s_mask + p * MASK_STRIDE)[lane] & inb) : 0u;
        mtn = act ? (reinterpret_cast<const uint32_t *>(s_mask + NP * MASK_STRIDE)[lane] & inb) : 0u;
        strct = act ? (reinterpret_cast<const uint32_t *>(s_mask + (NP + 1) * MASK_STRIDE)[lane] & inb) : 0u;
        a2 = act ? (reinterpret_cast<const uint32_t *>(s_mask + (NP + 2) * MASK_STRIDE)[lane] & inb) : 0u;
        __syncwarp();
    };

    // ---------------------------------------------------------------- a7: full recount (rare paths)
    auto recount = [&]() {
        __syncwarp();
        int acc[NP];
#pragma unroll
        for (int p = 0; p < NP; ++p) acc[p] = 0;
        for (int c = lane; c < HW; c += 32) {
            const int o = s_owner[c], a = s_army[c];
#pragma unroll
            for (int p = 0; p < NP; ++p) acc[p] += (o == p) ? a : 0;
        }
#pragma unroll
        for (int p = 0; p < NP; ++p) tot[p] = __reduce_add_sync(FULL, acc[p]);
    };

    // ---------------------------------------------------------------- a1: generator (R13, R14, R29, R30)
    auto generate = [&]() {
        __syncwarp();
        // clear: neutral empty plain; stride padding reads as mountain
        for (int i = lane; i < S / 4; i += 32) {
            reinterpret_cast<uint32_t *>(s_owner)[i] = 0xFFFFFFFFu;
            uint32_t tw = 0;
#pragma unroll
            for (int b = 0; b < 4; ++b) tw |= (4 * i + b >= HW) ? (uint32_t)T_MOUNTAIN << (8 * b) : 0u;
            reinterpret_cast<uint32_t *>(s_terr)[i] = tw;
            reinterpret_cast<uint32_t *>(s_army)[2 * i] = 0;
            reinterpret_cast<uint32_t *>(s_army)[2 * i + 1] = 0;
        }
        __syncwarp();
        uint32_t w[4];
        // (1) spawn distance window
        int lo = kp.dmin, hi = kp.dmax > 0 ? kp.dmax : 64;
        if (kp.spawn_exact) {
            philox(0, gid, episode, DOM_SPAWN << 24, kp.key0, kp.key1, w);
            lo = hi = kp.dmin + (int)mulhi32(w[1], (uint32_t)(kp.dmax - kp.dmin + 1));
        }
        // (3) mountains first (general cells are exempt: they are overwritten below and the city
        // draw only looks at PLAIN cells, so the order does not change the result)
        for (int q = lane; q < (HW + 3) / 4; q += 32) {
            philox((uint32_t)q, gid, episode, DOM_MOUNTAIN << 24, kp.key0, kp.key1, w);
            uint32_t tw = 0;
#pragma unroll
            for (int b = 0; b < 4; ++b)
                tw |= (w[b] < kp.mountain_thr || 4 * q + b >= HW) ? (uint32_t)T_MOUNTAIN << (8 * b) : 0u;
            reinterpret_cast<uint32_t *>(s_terr)[q] = tw;
        }
        __syncwarp();
        // (2) generals, one after the other
        int gr[NP], gc[NP];
#pragma unroll
        for (int p = 0; p < NP; ++p) { gr[p] = 0; gc[p] = 0; }
        for (int p = 0; p < P; ++p) {
            philox((uint32_t)p, gid, episode, DOM_SPAWN << 24, kp.key0, kp.key1, w);
            int cell;
            if (p == 0) {
                cell = (int)mulhi32(w[0], (uint32_t)HW);
            } else {
                int l = lo, h = hi;
                uint32_t cand, n;
                for (;;) {
                    cand = 0;
                    for (int j = 0; j < NW; ++j) {
                        const int c = 32 * j + (int)lane;
                        const int r = (int)(((uint32_t)c * kp.recipW) >> 16), col = c - r * W;
                        int mind = 1 << 20;
#pragma unroll
                        for (int q = 0; q < NP; ++q)
                            if (q < p) mind = min(mind, abs(r - gr[q]) + abs(col - gc[q]));
                        const uint32_t bal = __ballot_sync(FULL, c < HW && mind >= l && mind <= h && mind > 0);
                        if ((int)lane == j) cand = bal;
                    }
                    n = __reduce_add_sync(FULL, __popc(cand));
                    if (n > 0) break;
                    if (l > 0) l -= 1;
                    h += 1;
                }
                cell = select_kth(cand, mulhi32(w[0], n), lane);
            }
            const int r = (int)(((uint32_t)cell * kp.recipW) >> 16);
#pragma unroll
            for (int q = 0; q < NP; ++q)
                if (q == p) { gr[q] = r; gc[q] = cell - r * W; }
            if (lane == 0) {
                s_terr[cell] = (int8_t)T_GENERAL;
                s_owner[cell] = (int8_t)p;
                s_army[cell] = 1;
                B.general_cell[(size_t)g * P + p] = (int16_t)cell;
            }
        }
        __syncwarp();
        // (4) cities, one at a time, uniform over the remaining PLAIN cells
        uint32_t plain = 0;
        for (int j = 0; j < NW; ++j) {
            const int c = 32 * j + (int)lane;
            const uint32_t bal = __ballot_sync(FULL, c < HW && s_terr[c] == T_PLAIN);
            if ((int)lane == j) plain = bal;
        }
        uint32_t n = __reduce_add_sync(FULL, __popc(plain));
        for (int k = 0; k < kp.n_cities && n > 0; ++k, --n) {
            philox((uint32_t)k, gid, episode, DOM_CITY << 24, kp.key0, kp.key1, w);
            const int cell = select_kth(plain, mulhi32(w[0], n), lane);
            if ((int)lane == (cell >> 5)) plain &= ~(1u << (cell & 31));
            if (lane == 0) {
                s_terr[cell] = (int8_t)T_CITY;
                s_army[cell] = (int16_t)(kp.city_lo + (int)mulhi32(w[1], (uint32_t)kp.city_span));
            }
        }
        turn = 0;
        alive = allp;
        terrain_dirty = true;
#pragma unroll
        for (int p = 0; p < NP; ++p) tot[p] = (p < P) ? 1 : 0;
        __syncwarp();
    };

    // ---------------------------------------------------------------- load
    if (flags & F_RESET) {
        episode = (flags & F_KEEP_EPISODE) ? B.episode[g] : 0u;
        generate();
        if (lane == 0) {
            B.episode[g] = episode;
            B.episodes_done[g] = 0; B.truncations[g] = 0; B.sat_events[g] = 0;
            for (int p = 0; p < P; ++p) B.wins[(size_t)g * P + p] = 0;
        }
    } else {
        const uint4 *ga = reinterpret_cast<const uint4 *>(B.army + (size_t)g * S);
        const uint4 *go = reinterpret_cast<const uint4 *>(B.owner + (size_t)g * S);
        const uint4 *gt = reinterpret_cast<const uint4 *>(B.terrain + (size_t)g * S);
        const int n16 = S / 16;
        for (int i = lane; i < 4 * n16; i += 32) {
            const uint4 *src = (i < 2 * n16) ? ga + i : (i < 3 * n16 ? go + (i - 2 * n16) : gt + (i - 3 * n16));
            const uint32_t dst = (uint32_t)__cvta_generic_to_shared(wb + 16 * i);
            asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(dst), "l"(__cvta_generic_to_global(src)) : "memory");
        }
        turn = B.turn[g];
        alive = B.alive[g];
        done = B.done[g];
        winner = B.winner[g];
        episode = B.episode[g];
#pragma unroll
        for (int p = 0; p < NP; ++p)
            if (p < P) tot[p] = B.army_total[(size_t)g * P + p];
        if ((flags & F_DIGEST) && B.obs_digest) digest = B.obs_digest[g];
        asm volatile("cp.async.wait_all;\n" ::: "memory");
    }
    build_masks();
    if (flags & F_OBSERVE_ONLY) recount();

    // ---------------------------------------------------------------- a12: valid-action sampler (R24, R25)
    // returns this lane's action for player (lane) in act_l (lanes >= P hold 0)
    auto sample = [&](uint32_t gstep) -> int {
        uint32_t w[4];
        philox(0u, gid, gstep, (DOM_ACTION << 24) | (lane & 7u), kp.key0, kp.key1, w);
        // passable-target masks shared by all players: bit c says "the neighbour of c in direction d
        // exists and is not a mountain"
        const uint32_t pass = ~mtn & inb;
        uint32_t T[4];
        T[0] = bb_shl(pass, W, lane);             // up:    c - W
        T[1] = bb_shr(pass, W, lane);             // down:  c + W
        T[2] = bb_shl(pass, 1, lane) & notcol0;   // left:  c - 1
        T[3] = bb_shr(pass, 1, lane) & notcolL;   // right: c + 1
        int act_l = 0;
        for (int p = 0; p < P; ++p) {
            const uint32_t w0 = __shfl_sync(FULL, w[0], p), w1 = __shfl_sync(FULL, w[1], p);
            const uint32_t w2 = __shfl_sync(FULL, w[2], p), w3 = __shfl_sync(FULL, w[3], p);
            if (w0 < kp.pass_thr) continue;
            const uint32_t M = sel<NP>(own, p) & a2;
            uint32_t v[4];
#pragma unroll
            for (int d = 0; d < 4; ++d) v[d] = M & T[d];
            const uint32_t packed = __popc(v[0]) | (__popc(v[1]) << 16);
            const uint32_t packed2 = __popc(v[2]) | (__popc(v[3]) << 16);
            const uint32_t s01 = __reduce_add_sync(FULL, packed), s23 = __reduce_add_sync(FULL, packed2);
            uint32_t n[4] = {s01 & 0xFFFFu, s01 >> 16, s23 & 0xFFFFu, s23 >> 16};
            uint32_t total = n[0] + n[1] + n[2] + n[3];
            if (total == 0) continue;
            if (w3 < kp.bias_thr) {
                // largest owned stack, ties -> lowest cell index
                uint32_t best = 0, m = sel<NP>(own, p);
                while (m) {
                    const int b = __ffs(m) - 1;
                    m &= m - 1;
                    const uint32_t c = 32u * lane + (uint32_t)b;
                    best = max(best, ((uint32_t)(uint16_t)s_army[c] << 16) | (0xFFFFu - c));
                }
                best = __reduce_max_sync(FULL, best);
                const int bc = (int)(0xFFFFu - (best & 0xFFFFu));
                uint32_t nb = 0;
                uint32_t vb[4];
#pragma unroll
                for (int d = 0; d < 4; ++d) {
                    vb[d] = ((int)lane == (bc >> 5)) ? (v[d] & (1u << (bc & 31))) : 0u;
                    nb += __shfl_sync(FULL, vb[d], bc >> 5) ? 1u : 0u;
                }
                if (nb > 0) {
                    total = nb;
#pragma unroll
                    for (int d = 0; d < 4; ++d) { v[d] = vb[d]; n[d] = __shfl_sync(FULL, vb[d], bc >> 5) ? 1u : 0u; }
                }
            }
            uint32_t idx = mulhi32(w1, total);
            int d = 0;
            if (idx >= n[0]) { idx -= n[0]; d = 1;
                if (idx >= n[1]) { idx -= n[1]; d = 2;
                    if (idx >= n[2]) { idx -= n[2]; d = 3; } } }
            const uint32_t vd = d == 0 ? v[0] : (d == 1 ? v[1] : (d == 2 ? v[2] : v[3]));
            const int cell = select_kth(vd, idx, lane);
            const int a = cell * 9 + 1 + 2 * d + ((w2 < kp.half_thr) ? 1 : 0);
            if ((int)lane == p) act_l = a;
        }
        return act_l;
    };

    if (flags & F_SAMPLE_ONLY) {
        const bool frozen = !kp.auto_reset && done != 0;
        const int a = frozen ? 0 : sample(kp.global_step0);
        if ((int)lane < P) kp.sample_out[(size_t)g * P + lane] = a;
        return;
    }

    // ---------------------------------------------------------------- a10 + a11: fog of war and planes
    auto compute_vis = [&]() {
        __syncwarp();
        for (int p = 0; p < P; ++p) {
            uint32_t tm = 0;
            if (kp.team_size == 1) {
                tm = sel<NP>(own, p);
            } else {
                const uint32_t members = team_mask(p);
#pragma unroll
                for (int q = 0; q < NP; ++q) tm |= ((members >> q) & 1u) ? own[q] : 0u;
            }
            const uint32_t hz = tm | (bb_shl(tm, 1, lane) & notcol0) | (bb_shr(tm, 1, lane) & notcolL);
            const uint32_t vz = (hz | bb_shl(hz, W, lane) | bb_shr(hz, W, lane)) & inb;
            reinterpret_cast<uint32_t *>(s_mask + p * MASK_STRIDE)[lane] = vz;
        }
        __syncwarp();
    };

    auto emit_planes = [&](size_t slot) {
        const size_t base = (slot * (size_t)kp.N + (size_t)g) * (size_t)P * (size_t)S;
        int ch = (int)lane, p = 0;
        while (ch >= NC8) { ch -= NC8; ++p; }
        while (p < P) {
            const uint32_t vb = s_mask[p * MASK_STRIDE + ch];
            const uint4 a = *reinterpret_cast<const uint4 *>(s_army + 8 * ch);
            const uint2 o = *reinterpret_cast<const uint2 *>(s_owner + 8 * ch);
            const uint2 t = *reinterpret_cast<const uint2 *>(s_terr + 8 * ch);
            const uint32_t m0 = nib_to_bytes(vb & 15u), m1 = nib_to_bytes(vb >> 4);
            uint4 oa;
            oa.x = a.x & __byte_perm(m0, 0, 0x1100); oa.y = a.y & __byte_perm(m0, 0, 0x3322);
            oa.z = a.z & __byte_perm(m1, 0, 0x1100); oa.w = a.w & __byte_perm(m1, 0, 0x3322);
            uint2 oo, ot, ov;
            oo.x = (o.x & m0) | (~m0 & 0xFEFEFEFEu); oo.y = (o.y & m1) | (~m1 & 0xFEFEFEFEu);
            ot.x = (t.x & m0) | (~m0 & 0x04040404u); ot.y = (t.y & m1) | (~m1 & 0x04040404u);
            ov.x = m0 & 0x01010101u; ov.y = m1 & 0x01010101u;
            const size_t off = base + (size_t)p * S + 8 * (size_t)ch;
            __stcs(reinterpret_cast<uint4 *>(B.obs_army + off), oa);
            __stcs(reinterpret_cast<uint2 *>(B.obs_owner + off), oo);
            __stcs(reinterpret_cast<uint2 *>(B.obs_terrain + off), ot);
            __stcs(reinterpret_cast<uint2 *>(B.obs_vis + off), ov);
            ch += 32;
            while (ch >= NC8) { ch -= NC8; ++p; }
        }
    };

    // R28: h_p = sum_c pack(p, c) * key(c), pack = army | (owner + 2) << 16 | terrain << 20 | vis << 24.
    // A fogged cell packs to 0x400000, a visible one to x | 0x1000000, so
    // pack - 0x400000 = vis ? (x | 0xC00000) : 0 (terrain <= 3 leaves bits 22, 23 clear) and
    // h_p = 0x400000 * sum(key) + sum_c vismask & (x | 0xC00000) * key(c).
    auto chain_digest = [&](int rew_bits) {
        uint64_t ksum = 0;
        uint64_t h[NP];
#pragma unroll
        for (int p = 0; p < NP; ++p) h[p] = 0;
        for (int ch = lane; ch < NC8; ch += 32) {
            const uint4 a = *reinterpret_cast<const uint4 *>(s_army + 8 * ch);
            const uint2 o = *reinterpret_cast<const uint2 *>(s_owner + 8 * ch);
            const uint2 t = *reinterpret_cast<const uint2 *>(s_terr + 8 * ch);
            // per byte: (owner + 2) | terrain << 4
            const uint32_t otx = (((o.x & 0x0F0F0F0Fu) + 0x02020202u) & 0x0F0F0F0Fu) | (t.x << 4);
            const uint32_t oty = (((o.y & 0x0F0F0F0Fu) + 0x02020202u) & 0x0F0F0F0Fu) | (t.y << 4);
            const uint32_t aw[4] = {a.x, a.y, a.z, a.w};
            uint32_t vb[NP];
#pragma unroll
            for (int p = 0; p < NP; ++p) vb[p] = (p < P) ? s_mask[p * MASK_STRIDE + ch] : 0u;
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const uint32_t half = (i & 1) ? (aw[i >> 1] >> 16) : (aw[i >> 1] & 0xFFFFu);
                const uint32_t ob = (((i < 4) ? otx : oty) >> (8 * (i & 3))) & 0xFFu;
                const uint32_t x = half | (ob << 16) | 0xC00000u;
                const uint64_t key = s_key[8 * ch + i];
                ksum += key;
#pragma unroll
                for (int p = 0; p < NP; ++p)
                    if (p < P && ((vb[p] >> i) & 1u)) h[p] += (uint64_t)x * key;
            }
        }
        auto wsum = [&](uint64_t v) -> uint64_t {
#pragma unroll
            for (int o = 16; o >= 1; o >>= 1) v += __shfl_xor_sync(FULL, v, o);
            return v;
        };
        const uint64_t c0 = 0x400000ull * wsum(ksum);
        for (int p = 0; p < P; ++p) {
            uint64_t hp = 0;
#pragma unroll
            for (int q = 0; q < NP; ++q) hp = (q == p) ? h[q] : hp;
            digest = mix64(digest ^ (c0 + wsum(hp)));
        }
        const uint64_t tail = (uint64_t)done | ((uint64_t)(uint8_t)(winner + 2) << 8) | ((uint64_t)(uint32_t)rew_bits << 16);
        digest = mix64(digest ^ tail);
    };

    // growth of the cells in `m` (this lane's word): +1 saturating at 32767 (R21); returns saturations
    auto grow = [&](uint32_t m) -> int {
        int sat = 0;
        while (m) {
            const int b = __ffs(m) - 1;
            m &= m - 1;
            const int c = 32 * (int)lane + b;
            const int a = s_army[c];
            if (a >= 32767) { ++sat; }
            else {
                s_army[c] = (int16_t)(a + 1);
                if (a + 1 == 2) a2 |= 1u << b;
            }
        }
        return sat;
    };

    auto set_bit = [&](uint32_t &word, int c, bool on) {
        if ((int)lane == (c >> 5)) word = on ? (word | (1u << (c & 31))) : (word & ~(1u << (c & 31)));
    };

    // ================================================================ K turns
    const bool every = (flags & F_OBS_EVERY) != 0;
    for (int k = 0; k < kp.K; ++k) {
        const size_t slot = every ? (size_t)k : 0;
        const uint32_t gstep = kp.global_step0 + (uint32_t)k;
        const bool frozen = !kp.auto_reset && done != 0;  // R31
        int act_l = 0;
        if (!frozen) {
            if (flags & F_SAMPLER) act_l = sample(gstep);
            else if ((int)lane < P) act_l = kp.actions[(size_t)g * P + lane];
        }
        if (B.actions_out && (int)lane < P) B.actions_out[(slot * kp.N + g) * P + lane] = act_l;
        int rew_bits = 0;  // (reward[p] + 1) << 2p
        int rew[NP];
#pragma unroll
        for (int p = 0; p < NP; ++p) rew[p] = 0;

        if (!frozen) {
            bool need_recount = false;
            int sat_total = 0;
            // ---- a2 + a3: moves in ascending player index, each re-validated on the current board (R6, R7)
            const int first = (kp.rule_flags & GEN_RULE_ROTATE_PRIORITY) ? (turn % P) : 0;
            for (int i = 0; i < P; ++i) {
                int p = first + i;
                if (p >= P) p -= P;
                const int a = __shfl_sync(FULL, act_l, p);
                if (a <= 0 || a >= 9 * HW) continue;
                const int cell = a / 9, kk = a - 9 * cell;
                if (kk == 0) continue;
                const int dir = (kk - 1) >> 1, half = (kk - 1) & 1;
                const int r = (int)(((uint32_t)cell * kp.recipW) >> 16), col = cell - r * W;
                int dst;
                bool ok;
                if (dir == 0) { dst = cell - W; ok = r > 0; }
                else if (dir == 1) { dst = cell + W; ok = r < H - 1; }
                else if (dir == 2) { dst = cell - 1; ok = col > 0; }
                else { dst = cell + 1; ok = col < W - 1; }
                if (!ok) continue;
                const int asrc = s_army[cell];
                if (s_owner[cell] != p || asrc < 2 || s_terr[dst] == T_MOUNTAIN) continue;
                const int m = half ? (asrc >> 1) : (asrc - 1);  // R4
                const int nsrc = asrc - m;
                const int t = s_owner[dst], d = s_army[dst];
                const bool dst_general = s_terr[dst] == T_GENERAL;
                int ndst, nown = t;
                bool captured = false;
                const bool ally = t >= 0 && t != p && ((team_mask(p) >> t) & 1u);
                if (t == p || ally) {  // R8 / P:L97, R19
                    ndst = d + m;
                    if (ndst > 32767) { ndst = 32767; ++sat_total; need_recount = true; }
                    if (ally) {
                        if (!dst_general) {
                            nown = p;
#pragma unroll
                            for (int q = 0; q < NP; ++q) { if (q == p) tot[q] += d; if (q == t) tot[q] -= d; }
                        } else {
#pragma unroll
                            for (int q = 0; q < NP; ++q) { if (q == p) tot[q] -= m; if (q == t) tot[q] += m; }
                        }
                    }
                } else if (m > d) {
                    ndst = m - d;
                    nown = p;
                    captured = dst_general && t >= 0;  // R11, R12
#pragma unroll
                    for (int q = 0; q < NP; ++q) { if (q == p) tot[q] -= d; if (q == t) tot[q] -= d; }
                } else {
                    ndst = d - m;  // tie -> 0, previous owner keeps the cell
#pragma unroll
                    for (int q = 0; q < NP; ++q) { if (q == p) tot[q] -= m; if (q == t) tot[q] -= m; }
                }
                __syncwarp();
                if (lane == 0) {
                    s_army[cell] = (int16_t)nsrc;
                    s_army[dst] = (int16_t)ndst;
                    s_owner[dst] = (int8_t)nown;
                    if (captured) s_terr[dst] = (int8_t)T_CITY;
                }
                set_bit(a2, cell, nsrc >= 2);
                set_bit(a2, dst, ndst >= 2);
                if (nown != t) {
#pragma unroll
                    for (int q = 0; q < NP; ++q) {
                        if (q == nown) set_bit(own[q], dst, true);
                        if (q == t) set_bit(own[q], dst, false);
                    }
                }
                __syncwarp();
                if (captured) {  // a4: land transfer (R11)
                    const int q = t;
                    alive &= ~(1u << q);
                    if (lane == 0) B.general_cell[(size_t)g * P + q] = -1;
                    terrain_dirty = true;
                    need_recount = true;
                    const bool fl = (kp.rule_flags & GEN_RULE_CAPTURE_HALF_FLOOR) != 0;
                    for (int j = 0; j < NW; ++j) {
                        const int c = 32 * j + (int)lane;
                        bool ge2 = false;
                        if (c < HW) {
                            int av = s_army[c];
                            if (s_owner[c] == q) {
                                s_owner[c] = (int8_t)p;
                                av = fl ? (av >> 1) : ((av + 1) >> 1);
                                s_army[c] = (int16_t)av;
                            }
                            ge2 = av >= 2;
                        }
                        const uint32_t bal = __ballot_sync(FULL, ge2);
                        if ((int)lane == j) a2 = bal;
                    }
                    const uint32_t oq = sel<NP>(own, q);
#pragma unroll
                    for (int x = 0; x < NP; ++x) { if (x == p) own[x] |= oq; if (x == q) own[x] = 0; }
                    __syncwarp();
                }
            }
            // ---- a6: turn counter, then growth (R1, R2, R3)
            turn += 1;
            uint32_t owned = 0;
#pragma unroll
            for (int p = 0; p < NP; ++p) owned |= own[p];
            int sat_l = 0;
            const bool even = (turn & 1) == 0, tick = (turn % 50) == 0;
            if (even) {
                const uint32_t gm = strct & owned;
                sat_l += grow(gm);
                // structures are a handful of cells: one packed REDUX per pair of players
#pragma unroll
                for (int p = 0; p < NP; p += 2) {
                    if (p < P) {
                        const uint32_t s = __reduce_add_sync(FULL, __popc(gm & own[p]) | (__popc(gm & own[p + 1 < NP ? p + 1 : p]) << 16));
                        tot[p] += (int)(s & 0xFFFFu);
                        if (p + 1 < NP) tot[p + 1] += (int)(s >> 16);
                    }
                }
            }
            if (tick) {
                const uint32_t gm = (kp.rule_flags & GEN_RULE_TICK_PLAIN_ONLY) ? (owned & ~strct) : owned;
                sat_l += grow(gm);
#pragma unroll
                for (int p = 0; p < NP; p += 2) {
                    if (p < P) {
                        const uint32_t s = __reduce_add_sync(FULL, __popc(gm & own[p]) | (__popc(gm & own[p + 1 < NP ? p + 1 : p]) << 16));
                        tot[p] += (int)(s & 0xFFFFu);
                        if (p + 1 < NP) tot[p + 1] += (int)(s >> 16);
                    }
                }
            }
            if (even || tick) {
                const int s = __reduce_add_sync(FULL, sat_l);
                if (s) { sat_total += s; need_recount = true; }
                __syncwarp();
            }
            if (sat_total && lane == 0) B.sat_events[g] += (uint32_t)sat_total;
            if (need_recount) recount();
            // ---- a8: termination, reward, done (R16, R20)
            int living = 0, last = -1;
            for (int t = 0; t < kp.n_teams; ++t) {
                const uint32_t tm = (((1u << kp.team_size) - 1u) << (t * kp.team_size)) & allp;
                if (alive & tm) { ++living; last = t; }
            }
            const bool terminated = living <= 1;
            const bool truncated = !terminated && kp.max_turns > 0 && turn >= kp.max_turns;
            done = (terminated ? 1u : 0u) | (truncated ? 2u : 0u);
            winner = terminated ? last : -1;
            if (terminated) {
#pragma unroll
                for (int p = 0; p < NP; ++p)
                    if (p < P) rew[p] = (p / kp.team_size == last) ? 1 : -1;
            }
            if (done && lane == 0) {
                B.episodes_done[g] += 1;
                if (truncated) B.truncations[g] += 1;
                if (terminated)
                    for (int p = 0; p < P; ++p)
                        if (p / kp.team_size == last) B.wins[(size_t)g * P + p] += 1;
            }
        }
#pragma unroll
        for (int p = 0; p < NP; ++p)
            if (p < P) rew_bits |= (rew[p] + 1) << (2 * p);
        // outputs of this step
        const bool last_step = (k == kp.K - 1);
        if (every || last_step) {
            if ((int)lane < P) {
                int rv = 0;
#pragma unroll
                for (int p = 0; p < NP; ++p) rv = ((int)lane == p) ? rew[p] : rv;
                B.reward[(slot * kp.N + g) * P + lane] = (int8_t)rv;
            }
            if (lane == 0) {
                B.done[slot * kp.N + g] = (uint8_t)done;
                B.winner[slot * kp.N + g] = (int8_t)winner;
            }
        }
        // ---- a9: auto-reset (R17): reward / done describe the finished episode, state + obs the new one
        if (!frozen && done && kp.auto_reset) {
            episode += 1;
            if (lane == 0) B.episode[g] = episode;
            generate();
            build_masks();
        }
        // ---- a10 + a11 (R32: the state at the end of the call)
        const bool planes = (flags & F_OBS_PLANES) && (every || last_step);
        if (planes || (flags & F_DIGEST)) compute_vis();
        if (planes) emit_planes(slot);
        if ((flags & F_DIGEST) && !frozen) chain_digest(rew_bits);
    }

    if (kp.K == 0) {  // gen_reset / gen_observe: observation of the state as it stands
        if (flags & F_RESET) { done = 0; winner = -1; }
        compute_vis();
        if (flags & F_OBS_PLANES) emit_planes(0);
        if (flags & F_RESET) {
            if ((int)lane < P) B.reward[(size_t)g * P + lane] = 0;
            if (lane == 0) { B.done[g] = 0; B.winner[g] = -1; }
            if (flags & F_DIGEST) {
                int rb = 0;
                for (int p = 0; p < P; ++p) rb |= 1 << (2 * p);
                digest = 0;
                chain_digest(rb);
            }
        }
    }

    // ---------------------------------------------------------------- store state
    __syncwarp();
    {
        uint4 *ga = reinterpret_cast<uint4 *>(B.army + (size_t)g * S);
        uint2 *go = reinterpret_cast<uint2 *>(B.owner + (size_t)g * S);
        uint2 *gt = reinterpret_cast<uint2 *>(B.terrain + (size_t)g * S);
        for (int ch = lane; ch < NC8; ch += 32) {
            ga[ch] = *reinterpret_cast<const uint4 *>(s_army + 8 * ch);
            go[ch] = *reinterpret_cast<const uint2 *>(s_owner + 8 * ch);
            if (terrain_dirty) gt[ch] = *reinterpret_cast<const uint2 *>(s_terr + 8 * ch);
        }
        // land = popcount of the ownership bitboards (R23)
        int land_l = 0, tot_l = 0;
#pragma unroll
        for (int p = 0; p < NP; ++p) {
            const int l = __reduce_add_sync(FULL, __popc(own[p]));
            if ((int)lane == p) { land_l = l; tot_l = tot[p]; }
        }
        if ((int)lane < P) {
            B.land[(size_t)g * P + lane] = land_l;
            B.army_total[(size_t)g * P + lane] = tot_l;
        }
        if (lane == 0) {
            B.turn[g] = turn;
            B.alive[g] = (uint8_t)alive;
            if ((flags & F_DIGEST) && B.obs_digest) B.obs_digest[g] = digest;
        }
    }
}

}  // namespace gen
