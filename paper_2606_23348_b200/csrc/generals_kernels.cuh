// generals_kernels.cuh -- device code of the batched Generals.io step for sm_100a.
//
// WARP-AUTONOMOUS design.  A warp owns GW = 4 consecutive games; an OCTET of 8 lanes owns one game
// from load to store.  The warp's three state planes (int16 army, int8 owner, int8 terrain of its 4
// games) are contiguous in HBM and are staged in the warp's own slice of shared memory with three TMA
// bulk copies (cp.async.bulk + the warp's own mbarrier).  After one CTA barrier in the prologue (small
// constant tables) no warp ever waits for another one: phases are separated by __syncwarp() only, so
// while one warp waits for its loads or drains its observation stores the others compute.
//
//   * CELL passes -- the octet walks its board in 8-cell chunks (lane l: chunks l, l+8, ...) with
//     SIMD-in-register byte arithmetic and 16 / 8-byte shared and global accesses: bitboard
//     construction, tick growth, observation planes (the dominant HBM traffic, full-sector streaming
//     stores), observation digest.
//   * WORD passes -- flat bitboards (one bit per cell, word j = cells 32j..32j+31: own[p], structure,
//     army >= 2, the four static "target is free" rows, vis[p]) live in shared memory.  The octet is
//     split by player: LPP = 8 / NP lanes serve one (game, player) pair and each of them streams
//     through WS consecutive words: Philox valid-action sampler (popcount enumeration, scan over the
//     LPP lanes), fog-of-war dilation (funnel shifts, sliding window).  All players advance in the
//     same instruction stream.
//   * SERIAL passes -- lane 0 of the octet runs the scalar rules: move / combat / capture,
//     termination, reward; four games advance per warp instruction.
//
// Rare heavy paths (board generation at reset: the whole warp per game; general capture with land
// transfer; int16 saturation) never tax the common path.
//
// Rules: PAPER.md section IV, readings R1..R32 of DESIGN.md.  This file shares nothing
// with oracle/ (the CPU checker); it is written from the same rules text.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "generals.h"

// `if constexpr (OFFICIAL) { ...; return; }` leaves the synthetic generator behind it unreachable in the official
// instantiations: that is the intent, not a finding
#pragma nv_diag_suppress 128

namespace gen {

constexpr uint32_t FULL = 0xffffffffu;
constexpr int LPG = 8;            // lanes per game: the octet
constexpr int GW = 32 / LPG;      // games per warp

enum : uint32_t {
    F_RESET = 1u << 0,         // generate every board first (gen_reset)
    F_SAMPLER = 1u << 1,       // draw actions with the built-in sampler
    F_OBS_PLANES = 1u << 2,    // write observation planes
    F_OBS_EVERY = 1u << 3,     // ... for every step, slot k
    F_DIGEST = 1u << 4,        // chain the observation digest
    F_OBSERVE_ONLY = 1u << 5,  // gen_observe: recount + planes, no turn
    F_SAMPLE_ONLY = 1u << 6,   // gen_sample: actions only
    F_KEEP_EPISODE = 1u << 7,
    F_RUNTIME = 0xFFFFFFFFu,   // template argument FF: read the flags word from KParams (generic kernel)
    F_K1 = 1u << 30,           // template argument FF only: exactly one turn per launch (gen_step)
};

enum : int { T_PLAIN = 0, T_MOUNTAIN = 1, T_CITY = 2, T_GENERAL = 3, T_FOG = 4 };

// per-game flags raised by the serial passes for the following parallel pass
enum : uint32_t {
    GF_REBUILD = 1u << 0,        // planes changed wholesale: rebuild the bitboards
    GF_RECOUNT = 1u << 1,        // recount army totals from the planes
    GF_RESET = 1u << 2,          // auto-reset: generate a new board
    GF_FROZEN = 1u << 3,         // finished game without auto-reset (R31)
    GF_TERRAIN_DIRTY = 1u << 4,  // terrain plane must be written back
    GF_GROW_EVEN = 1u << 5,      // structures of owned cells +1 this turn
    GF_GROW_TICK = 1u << 6,      // all owned cells +1 this turn
    GF_ALL_DIRTY = 1u << 7,      // write back the whole army / owner planes
};

// per-game scalars in shared memory
struct GameS {
    int32_t turn, winner;
    uint32_t alive, done, episode, flags, sat, dirtyO;  // dirtyO bit u: owner cells 32u..32u+31 changed
    uint32_t dirtyA[2];                                 // bit u: army cells 16u..16u+15 changed
    unsigned long long digest;
    int32_t tot[8], land[8], act[8];
    int32_t rew_bits, pad_;
};

struct KParams {
    int32_t N, H, W, P, HW, S, NW, NC8, NCH, RW, M, BW;  // BW: words per row of gen_buffers.bitboards
    int32_t team_size, n_teams;
    int32_t n_cities, city_lo, city_span;
    int32_t dmin, dmax, spawn_exact, max_turns, auto_reset;
    int32_t map_mode, n_cities_max, play_min, castle_radius;  // R36 (official generator)
    uint32_t rule_flags, gid_base, mountain_thr, key0, key1;
    uint32_t pass_thr, half_thr, bias_thr;
    uint32_t global_step0, flags, recipW;
    int32_t K, WPC;  // turns per launch; warps per CTA
    int32_t count;   // k_step: take a ticket per group of 4 games in gen_buffers.step_epoch and record completion
    int32_t chain;   // k_step: wait per warp for the earlier tickets of its group instead of for the previous grid
    int32_t stack_ok;  // k_step (BIAS): gen_buffers.stack_cache was written by this handle's previous launch for this step
    // shared memory: [tables | digest keys | warp 0 | warp 1 | ...]; w_* are offsets inside a warp's slice
    uint32_t off_key, off_warp0, warp_bytes, w_owner, w_terr, w_mask, w_game, w_bar, w_scratch, smem_bytes;
    unsigned long long key_sum;  // sum of the digest keys of cells 0..HW-1
    gen_buffers b;
    const int32_t *actions;
    int32_t *sample_out;
    // gen_step_host[_async] on k_step: every game's reward [P] and done are also written to these (device aliases of
    // pinned host arrays [N][P] / [N]; either may be NULL) by the lane that writes them to the device buffers
    int8_t *mirror_reward;
    uint8_t *mirror_done;
    uint32_t notcol0[32], notcolL[32], inb[32];  // column / in-bounds masks of bitboard word j
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

__device__ __forceinline__ uint32_t mulhi32(uint32_t u, uint32_t n) { return __umulhi(u, n); }

// Digest keys (R28): key(c) = the (c + 1)-th output of splitmix64(seed 0), forced odd.  They do not depend on the
// board, so they are a compile-time table in global memory, read through the read-only path (8 KB, L1-resident)
// instead of a per-CTA copy in shared memory (which cost the fused rollout one resident CTA per SM).
struct DigestKeys { unsigned long long k[1024]; };
constexpr DigestKeys make_digest_keys() {
    DigestKeys t{};
    for (int c = 0; c < 1024; ++c) {
        unsigned long long z = (unsigned long long)(c + 1) * 0x9E3779B97F4A7C15ull;
        z ^= z >> 30; z *= 0xBF58476D1CE4E5B9ull;
        z ^= z >> 27; z *= 0x94D049BB133111EBull;
        z ^= z >> 31;
        t.k[c] = z | 1ull;
    }
    return t;
}
static __device__ const DigestKeys g_digest_keys = make_digest_keys();

__device__ __forceinline__ int nth_bit(uint32_t w, uint32_t r) {  // position of the r-th (0-based) set bit
    int pos = 0;
#pragma unroll
    for (int s = 16; s >= 1; s >>= 1) {
        const uint32_t c = __popc((w >> pos) & ((1u << s) - 1u));
        if (r >= c) { r -= c; pos += s; }
    }
    return pos;
}

// warp-level: cell index of the k-th set bit (row-major) of a flat bitboard held one word per lane
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

// SIMD-in-register byte helpers
__device__ __forceinline__ uint32_t prmt(uint32_t a, uint32_t b, uint32_t sel) {
    uint32_t d;
    asm("prmt.b32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(sel));
    return d;
}
// 4 bits -> a word whose byte i has bit i of the nibble in its MSB (other bits are don't-care);
// prmt's sign-replicate selectors (8 | byte index) then expand it: 0xBA98 -> four 0x00 / 0xFF byte
// masks, 0x9988 / 0xBBAA -> the two int16-pair masks of cells (0, 1) / (2, 3).
__device__ __forceinline__ uint32_t nib_sign(uint32_t nib) { return nib * 0x10204080u; }
// Bit gathering.  x0 / x1 hold one flag per byte (cells 0..3 / 4..7) at bit position B; bit B + 4 of
// every byte must be clear, the other bits are don't-care.  nib8 moves them to bits 0, 4, ..., 28 (cell c < 4 at bit 8c, cell 4 + c at bit
// 8c + 4); one multiply then lines the eight flags up in the top byte.
template <int B>
__device__ __forceinline__ uint32_t gather8(uint32_t x0, uint32_t x1) {
    const uint32_t z = (B <= 4 ? ((x1 << (4 - B)) | (x0 >> B)) : ((x1 >> (B - 4)) | (x0 >> B))) & 0x11111111u;
    return (z * 0x01020408u) >> 24;
}
__device__ __forceinline__ uint32_t eq_bytes(uint32_t w, uint32_t pat) {  // 0x01 where byte == pat byte
    const uint32_t x = w ^ pat;
    const uint32_t y = ((x & 0x7F7F7F7Fu) + 0x7F7F7F7Fu) | x;
    return (~y >> 7) & 0x01010101u;
}
// 8 int16 armies (all in [0, 32767]) -> 8 bits "army >= 2": min(a, 2) has bit 1 set iff a >= 2
__device__ __forceinline__ uint32_t ge2_bits(const uint4 &a) {
    const uint32_t y0 = __vminu2(a.x, 0x00020002u), y1 = __vminu2(a.y, 0x00020002u);
    const uint32_t y2 = __vminu2(a.z, 0x00020002u), y3 = __vminu2(a.w, 0x00020002u);
    return gather8<1>(__byte_perm(y0, y1, 0x6420), __byte_perm(y2, y3, 0x6420));
}

// ------------------------------------------------------------------------------------------------
// mbarrier + TMA bulk copy (global -> shared), raw PTX
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(__cvta_generic_to_global(src)), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void l2_prefetch(const void *src, uint32_t bytes) {  // TMA bulk prefetch HBM -> L2
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(__cvta_generic_to_global(src)), "r"(bytes)
                 : "memory");
}
// programmatic dependent launch: let the next grid in the stream start being placed / wait until everything the
// previous grid wrote is visible
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    do {
        asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                     : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    } while (!ok);
}

// ------------------------------------------------------------------------------------------------
// NEXT-3: the official map generator (R36), one warp per game, 1v1.
// The board is held as ROW WORDS while it is built: lane r owns row r, bit c = column c (H, W <= 32).  Steps
// between cells (the paper's BFS distance) come from a frontier expansion on those words: one level = two
// shifts, two shuffles (the rows above and below) and a mask with the passable cells.
__device__ __forceinline__ uint32_t rows_count(uint32_t word) { return __reduce_add_sync(FULL, __popc(word)); }

// cell index of the k-th set bit, row-major, of a board held one row word per lane
__device__ __forceinline__ int rows_select(uint32_t word, uint32_t k, uint32_t lane, int W) {
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
    return j * W + nth_bit(wj, k - excl_j);
}

// V_i = the cells within t_i steps of (src_r, src_c) over `pass` (t_i < 0: the empty set); stops at the largest
// threshold or when the frontier dies (then every later threshold sees the whole reachable set)
static __device__ __noinline__ void rows_bfs(uint32_t pass, int src_r, int src_c, uint32_t lane, int t0, int t1, int t2,
                                      uint32_t &V0, uint32_t &V1, uint32_t &V2) {
    uint32_t V = ((int)lane == src_r) ? 1u << src_c : 0u, F = V;
    V0 = V1 = V2 = 0u;
    const int tmax = max(t0, max(t1, t2));
    for (int L = 0;; ++L) {
        if (L == t0) V0 = V;
        if (L == t1) V1 = V;
        if (L == t2) V2 = V;
        if (L >= tmax) break;
        uint32_t up = __shfl_up_sync(FULL, F, 1), dn = __shfl_down_sync(FULL, F, 1);
        if (lane == 0) up = 0u;
        if (lane == 31) dn = 0u;
        const uint32_t N = ((F << 1) | (F >> 1) | up | dn) & pass & ~V;
        if (!__any_sync(FULL, N != 0u)) {
            if (t0 > L) V0 = V;
            if (t1 > L) V1 = V;
            if (t2 > L) V2 = V;
            break;
        }
        V |= N;
        F = N;
    }
}

static __device__ __noinline__ void generate_official(const KParams &kp, uint32_t lane, uint32_t gid, uint32_t episode,
                                               int16_t *A, int8_t *O, int8_t *Tr, int16_t *gcell_out,
                                               int8_t *psize_out) {
    const int H = kp.H, W = kp.W, HW = kp.HW, S = kp.S;
    constexpr int kAttempts = 16, kFar = (1 << 20) - 1;
    uint32_t w[4];
    for (uint32_t a = 0; a < (uint32_t)kAttempts; ++a) {
        const bool last = a == (uint32_t)kAttempts - 1;
        __syncwarp();
        // (0) sizes of this attempt
        philox(0u, gid, episode, (DOM_SPAWN << 24) | a, kp.key0, kp.key1, w);
        int h = H, wd = W;
        if (kp.play_min > 0) {
            const int hmin = min(kp.play_min, H), wmin = min(kp.play_min, W);
            h = hmin + (int)mulhi32(w[0], (uint32_t)(H - hmin + 1));
            wd = wmin + (int)mulhi32(w[1], (uint32_t)(W - wmin + 1));
        }
        int lo = kp.dmin, hi = kp.dmax > 0 ? kp.dmax : kFar;
        if (kp.spawn_exact) lo = hi = kp.dmin + (int)mulhi32(w[2], (uint32_t)(kp.dmax - kp.dmin + 1));
        int n_castles = kp.n_cities;
        if (kp.n_cities_max > kp.n_cities) n_castles += (int)mulhi32(w[3], (uint32_t)(kp.n_cities_max - kp.n_cities + 1));
        // (1) terrain: mountains outside the playable rectangle, Bernoulli inside (none on the last attempt)
        for (int q = (int)lane; q < S / 4; q += 32) {
            philox((uint32_t)q, gid, episode, (DOM_MOUNTAIN << 24) | a, kp.key0, kp.key1, w);
            uint32_t tw = 0;
#pragma unroll
            for (int b = 0; b < 4; ++b) {
                const int c = 4 * q + b, r = (int)(((uint32_t)c * kp.recipW) >> 16), col = c - r * W;
                const bool playable = c < HW && r < h && col < wd;
                tw |= (!playable || (!last && w[b] < kp.mountain_thr)) ? (uint32_t)T_MOUNTAIN << (8 * b) : 0u;
            }
            reinterpret_cast<uint32_t *>(Tr)[q] = tw;
            reinterpret_cast<uint32_t *>(O)[q] = 0xFFFFFFFFu;
            reinterpret_cast<uint32_t *>(A)[2 * q] = 0;
            reinterpret_cast<uint32_t *>(A)[2 * q + 1] = 0;
        }
        __syncwarp();
        uint32_t plain = 0;                                     // lane r: the PLAIN cells of row r
        if ((int)lane < H)
            for (int col = 0; col < W; ++col) plain |= (uint32_t)(Tr[(int)lane * W + col] == T_PLAIN) << col;
        const uint32_t pass = plain;                            // non-mountain cells: castles do not block
        // (2) general 0
        philox(1u, gid, episode, (DOM_SPAWN << 24) | a, kp.key0, kp.key1, w);
        const uint32_t u_g1 = w[1];
        uint32_t n = rows_count(plain);
        if (n == 0) continue;
        const int g0 = rows_select(plain, mulhi32(w[0], n), lane, W);
        const int r0 = (int)(((uint32_t)g0 * kp.recipW) >> 16), c0 = g0 - r0 * W;
        if ((int)lane == r0) plain &= ~(1u << c0);
        // (3), (4) general 1 at lo..hi steps
        uint32_t cand, Vlo, Vhi, Vnear0, Vnear1, unused;
        for (;;) {
            rows_bfs(pass, r0, c0, lane, lo - 1, hi, kp.castle_radius, Vlo, Vhi, Vnear0);
            cand = plain & Vhi & ~Vlo;
            n = rows_count(cand);
            if (n > 0 || !last) break;
            if (lo == 0 && hi >= HW) break;
            if (lo > 0) lo -= 1;
            hi += 1;
        }
        if (n == 0) continue;
        const int g1 = rows_select(cand, mulhi32(u_g1, n), lane, W);
        const int r1 = (int)(((uint32_t)g1 * kp.recipW) >> 16), c1 = g1 - r1 * W;
        if ((int)lane == r1) plain &= ~(1u << c1);
        rows_bfs(pass, r1, c1, lane, kp.castle_radius, -1, -1, Vnear1, unused, unused);
        // (5) castles: the first near general 0, the second near general 1, the rest anywhere
        bool ok = true;
        for (int k = 0; k < n_castles; ++k) {
            const bool near = kp.castle_radius > 0 && k < 2;
            uint32_t set = near ? plain & (k == 0 ? Vnear0 : Vnear1) : 0u;
            n = near ? rows_count(set) : 0u;
            if (near && n == 0 && !last) { ok = false; break; }
            if (n == 0) { set = plain; n = rows_count(set); }
            if (n == 0) break;
            philox((uint32_t)k, gid, episode, (DOM_CITY << 24) | a, kp.key0, kp.key1, w);
            const int cell = rows_select(set, mulhi32(w[0], n), lane, W);
            const int rc = (int)(((uint32_t)cell * kp.recipW) >> 16);
            if ((int)lane == rc) plain &= ~(1u << (cell - rc * W));
            if (lane == 0) {
                Tr[cell] = (int8_t)T_CITY;
                A[cell] = (int16_t)(kp.city_lo + (int)mulhi32(w[1], (uint32_t)kp.city_span));
            }
        }
        if (!ok) continue;
        if (lane == 0) {
            Tr[g0] = (int8_t)T_GENERAL; O[g0] = 0; A[g0] = 1; gcell_out[0] = (int16_t)g0;
            Tr[g1] = (int8_t)T_GENERAL; O[g1] = 1; A[g1] = 1; gcell_out[1] = (int16_t)g1;
            if (psize_out) { psize_out[0] = (int8_t)h; psize_out[1] = (int8_t)wd; }
        }
        break;
    }
    __syncwarp();
}

// ------------------------------------------------------------------------------------------------
// a1: board generator (R13, R14, R29, R30), one warp per game, planes in shared memory (S cells each).
// Writes general_cell[p] through gcell_out.  Used by the per-step kernel (a call, not inlined: generation is rare
// and must not tax the register allocation of the turn); the staged kernel carries the same procedure inline.
template <int NP, bool OFFICIAL>
__device__ __noinline__ void generate_board(const KParams &kp, uint32_t lane, uint32_t gid, uint32_t episode,
                                            int16_t *A, int8_t *O, int8_t *Tr, int16_t *gcell_out, int8_t *psize_out) {
    const int P = kp.P, HW = kp.HW, S = kp.S, NW = kp.NW, W = kp.W;
    __syncwarp();
    if (!OFFICIAL && psize_out && lane == 0) { psize_out[0] = (int8_t)kp.H; psize_out[1] = (int8_t)kp.W; }
    if constexpr (OFFICIAL) {                                    // the official generator (R36)
        generate_official(kp, lane, gid, episode, A, O, Tr, gcell_out, psize_out);
        return;
    }
    for (int i = lane; i < S / 4; i += 32) {
        reinterpret_cast<uint32_t *>(O)[i] = 0xFFFFFFFFu;
        reinterpret_cast<uint32_t *>(A)[2 * i] = 0;
        reinterpret_cast<uint32_t *>(A)[2 * i + 1] = 0;
    }
    uint32_t w[4];
    int lo = kp.dmin, hi = kp.dmax > 0 ? kp.dmax : 64;
    if (kp.spawn_exact) {
        philox(0, gid, episode, DOM_SPAWN << 24, kp.key0, kp.key1, w);
        lo = hi = kp.dmin + (int)mulhi32(w[1], (uint32_t)(kp.dmax - kp.dmin + 1));
    }
    for (int q = lane; q < S / 4; q += 32) {
        philox((uint32_t)q, gid, episode, DOM_MOUNTAIN << 24, kp.key0, kp.key1, w);
        uint32_t tw = 0;
#pragma unroll
        for (int b = 0; b < 4; ++b)
            tw |= (w[b] < kp.mountain_thr || 4 * q + b >= HW) ? (uint32_t)T_MOUNTAIN << (8 * b) : 0u;
        reinterpret_cast<uint32_t *>(Tr)[q] = tw;
    }
    __syncwarp();
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
            Tr[cell] = (int8_t)T_GENERAL;
            O[cell] = (int8_t)p;
            A[cell] = 1;
            gcell_out[p] = (int16_t)cell;
        }
    }
    __syncwarp();
    uint32_t plain = 0;
    for (int j = 0; j < NW; ++j) {
        const int c = 32 * j + (int)lane;
        const uint32_t bal = __ballot_sync(FULL, c < HW && Tr[c] == T_PLAIN);
        if ((int)lane == j) plain = bal;
    }
    uint32_t n = __reduce_add_sync(FULL, __popc(plain));
    for (int k = 0; k < kp.n_cities && n > 0; ++k, --n) {
        philox((uint32_t)k, gid, episode, DOM_CITY << 24, kp.key0, kp.key1, w);
        const int cell = select_kth(plain, mulhi32(w[0], n), lane);
        if ((int)lane == (cell >> 5)) plain &= ~(1u << (cell & 31));
        if (lane == 0) {
            Tr[cell] = (int8_t)T_CITY;
            A[cell] = (int16_t)(kp.city_lo + (int)mulhi32(w[1], (uint32_t)kp.city_span));
        }
    }
    __syncwarp();
}

// ================================================================================================
// Template arguments: NP = bound of the player loops (register arrays).  CH x CW > 0 = the board size is a
// compile-time constant and P == NP exactly (the paper-sized configs: strides, word counts and the row
// division fold into immediates and the cell loops unroll); 0 = any board up to 32 x 32, read from KParams.
// FF = the mode flags as a compile-time constant (dead modes drop out of the instruction stream), or
// F_RUNTIME.  With FF fixed, F_SAMPLER alone stays a runtime choice.
template <int NP, int CH, int CW, uint32_t FF, bool OFFICIAL>
__global__ void __launch_bounds__(256) k_generals(const __grid_constant__ KParams kp) {
    constexpr bool FIXED = CH > 0;
    constexpr int LPP = LPG / NP;  // lanes serving one (game, player) pair in the word passes
    extern __shared__ __align__(128) unsigned char smem[];
    const int tid = threadIdx.x;
    const uint32_t lane = tid & 31u;
    const int wic = tid >> 5;
    const int ol = (int)(lane & (LPG - 1)), sub = (int)(lane / LPG);  // lane of the octet, game of the warp
    const uint32_t gmask = ((1u << LPG) - 1u) << (sub * LPG);         // the lanes of this octet
    const int pl = ol / LPP, sl = ol % LPP;                           // word passes: my player, my sub-lane
    constexpr int cHW = CH * CW, cS = (cHW + 15) / 16 * 16, cNW = (cHW + 31) / 32;
    const int H = FIXED ? CH : kp.H, W = FIXED ? CW : kp.W, P = FIXED ? NP : kp.P;
    const int HW = FIXED ? cHW : kp.HW, S = FIXED ? cS : kp.S, NW = FIXED ? cNW : kp.NW;
    const int NC8 = FIXED ? cS / 8 : kp.NC8, NCH = FIXED ? 4 * cNW : kp.NCH;
    const int RW = FIXED ? (cNW | 1) : kp.RW, M = FIXED ? 2 * NP + 7 : kp.M;
    const int BW = FIXED ? (cNW + 7) / 8 * 8 : kp.BW;
    const int WS = (NW + LPP - 1) / LPP;  // words per sub-lane
    const uint32_t flags = (FF == F_RUNTIME) ? kp.flags : ((FF & ~F_K1) | (kp.flags & F_SAMPLER));
    const int K = (FF != F_RUNTIME && (FF & F_K1)) ? 1 : kp.K;
    const gen_buffers &B = kp.b;
    const int wg0 = (blockIdx.x * kp.WPC + wic) * GW;  // first game of this warp
    const int nwg = min(GW, kp.N - wg0);               // games of this warp (<= 0: nothing to do)
    const bool gvalid = sub < nwg;
    const int g = wg0 + sub;
    const uint32_t allp = (1u << P) - 1u;
    const bool teams = (FIXED && NP == 2) ? false : kp.team_size > 1;

    // CTA-wide tables, index j + 1 for bitboard word j (entries 0 and 33 are zero guards): column masks,
    // in-bounds mask; digest keys
    uint32_t *s_nc0 = reinterpret_cast<uint32_t *>(smem) + 1, *s_ncL = s_nc0 + 34, *s_inb = s_nc0 + 68;
    // this warp's slice
    unsigned char *wb = smem + kp.off_warp0 + (size_t)wic * kp.warp_bytes;
    int16_t *s_army = reinterpret_cast<int16_t *>(wb);
    int8_t *s_owner = reinterpret_cast<int8_t *>(wb + kp.w_owner);
    int8_t *s_terr = reinterpret_cast<int8_t *>(wb + kp.w_terr);
    uint32_t *s_mask = reinterpret_cast<uint32_t *>(wb + kp.w_mask);
    GameS *s_game = reinterpret_cast<GameS *>(wb + kp.w_game);
    const uint32_t bar = smem_u32(wb + kp.w_bar);

    // bitboard rows of a game: own[0..P-1], structure (city / general), army >= 2, ok[4] (source cells whose
    // up / down / left / right target is on the board and no mountain: static per board), vis[0..P-1],
    // mountain (or off the board).
    const int R_STR = P, R_A2 = P + 1, R_OK = P + 2, R_VIS = P + 6, R_MTN = 2 * P + 6;
    auto mrow = [&](int m, int lg) -> uint32_t * { return s_mask + (lg * M + m) * RW; };
    auto mrow8 = [&](int m, int lg) -> unsigned char * { return reinterpret_cast<unsigned char *>(mrow(m, lg)); };

    auto team_mask = [&](int p) -> uint32_t {
        const int t = p / kp.team_size;
        return (((1u << kp.team_size) - 1u) << (t * kp.team_size)) & allp;
    };
    auto row_of = [&](int cell) -> int {
        return FIXED ? (int)((uint32_t)cell / (uint32_t)(FIXED ? CW : 1)) : (int)(((uint32_t)cell * kp.recipW) >> 16);
    };

    // ---------------------------------------------------------------- a1: generator, one warp per game
    // (R13, R14, R29, R30)
    auto generate = [&](int lg) {
        int16_t *A = s_army + (size_t)lg * S;
        int8_t *O = s_owner + (size_t)lg * S, *Tr = s_terr + (size_t)lg * S;
        GameS &gs = s_game[lg];
        const int gg = wg0 + lg;
        const uint32_t gid = kp.gid_base + (uint32_t)gg, episode = gs.episode;
        __syncwarp();
        if constexpr (OFFICIAL) {                                // R36, in the instantiations compiled for it
            generate_official(kp, lane, gid, episode, A, O, Tr, B.general_cell + (size_t)gg * P,
                              B.play_size ? B.play_size + 2 * (size_t)gg : nullptr);
            if (lane == 0) {
                gs.turn = 0;
                gs.alive = allp;
                gs.flags |= GF_TERRAIN_DIRTY | GF_ALL_DIRTY;
                for (int p = 0; p < P; ++p) { gs.tot[p] = 1; gs.land[p] = 1; }
            }
            __syncwarp();
            return;
        }
        if (B.play_size && lane == 0) { B.play_size[2 * (size_t)gg] = (int8_t)H; B.play_size[2 * (size_t)gg + 1] = (int8_t)W; }
        for (int i = lane; i < S / 4; i += 32) {
            reinterpret_cast<uint32_t *>(O)[i] = 0xFFFFFFFFu;
            reinterpret_cast<uint32_t *>(A)[2 * i] = 0;
            reinterpret_cast<uint32_t *>(A)[2 * i + 1] = 0;
        }
        uint32_t w[4];
        // (1) spawn distance window
        int lo = kp.dmin, hi = kp.dmax > 0 ? kp.dmax : 64;
        if (kp.spawn_exact) {
            philox(0, gid, episode, DOM_SPAWN << 24, kp.key0, kp.key1, w);
            lo = hi = kp.dmin + (int)mulhi32(w[1], (uint32_t)(kp.dmax - kp.dmin + 1));
        }
        // (3) mountains first (general cells are exempt: they are overwritten below and the city draw only
        // looks at PLAIN cells, so the order does not change the result); stride padding reads as mountain
        for (int q = lane; q < S / 4; q += 32) {
            philox((uint32_t)q, gid, episode, DOM_MOUNTAIN << 24, kp.key0, kp.key1, w);
            uint32_t tw = 0;
#pragma unroll
            for (int b = 0; b < 4; ++b)
                tw |= (w[b] < kp.mountain_thr || 4 * q + b >= HW) ? (uint32_t)T_MOUNTAIN << (8 * b) : 0u;
            reinterpret_cast<uint32_t *>(Tr)[q] = tw;
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
                        const int r = row_of(c), col = c - r * W;
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
            const int r = row_of(cell);
#pragma unroll
            for (int q = 0; q < NP; ++q)
                if (q == p) { gr[q] = r; gc[q] = cell - r * W; }
            if (lane == 0) {
                Tr[cell] = (int8_t)T_GENERAL;
                O[cell] = (int8_t)p;
                A[cell] = 1;
                B.general_cell[(size_t)gg * P + p] = (int16_t)cell;
            }
        }
        __syncwarp();
        // (4) cities, one at a time, uniform over the remaining PLAIN cells
        uint32_t plain = 0;
        for (int j = 0; j < NW; ++j) {
            const int c = 32 * j + (int)lane;
            const uint32_t bal = __ballot_sync(FULL, c < HW && Tr[c] == T_PLAIN);
            if ((int)lane == j) plain = bal;
        }
        uint32_t n = __reduce_add_sync(FULL, __popc(plain));
        for (int k = 0; k < kp.n_cities && n > 0; ++k, --n) {
            philox((uint32_t)k, gid, episode, DOM_CITY << 24, kp.key0, kp.key1, w);
            const int cell = select_kth(plain, mulhi32(w[0], n), lane);
            if ((int)lane == (cell >> 5)) plain &= ~(1u << (cell & 31));
            if (lane == 0) {
                Tr[cell] = (int8_t)T_CITY;
                A[cell] = (int16_t)(kp.city_lo + (int)mulhi32(w[1], (uint32_t)kp.city_span));
            }
        }
        if (lane == 0) {
            gs.turn = 0;
            gs.alive = allp;
            gs.flags |= GF_TERRAIN_DIRTY | GF_ALL_DIRTY;
            for (int p = 0; p < P; ++p) { gs.tot[p] = 1; gs.land[p] = 1; }
        }
        __syncwarp();
    };

    // ---------------------------------------------------------------- cell pass: bitboards of one game (octet)
    // chunk ch = cells 8ch..8ch+7 -> byte ch of the rows own[p], mountain, structure, army >= 2
    auto build_game = [&](int lg) {
        const unsigned char *sa = reinterpret_cast<const unsigned char *>(s_army + (size_t)lg * S);
        const unsigned char *so = reinterpret_cast<const unsigned char *>(s_owner + (size_t)lg * S);
        const unsigned char *st = reinterpret_cast<const unsigned char *>(s_terr + (size_t)lg * S);
        unsigned char *rows = mrow8(0, lg);
        const int rb = 4 * RW;  // row stride in bytes
#pragma unroll 3
        for (int ch = ol; ch < NC8; ch += LPG) {
            const uint2 o = *reinterpret_cast<const uint2 *>(so + 8 * ch);
            const uint2 t = *reinterpret_cast<const uint2 *>(st + 8 * ch);
            const uint4 a = *reinterpret_cast<const uint4 *>(sa + 16 * ch);
            if (NP == 2) {
                // owner in {-1, 0, 1}: bit 7 = neutral, bit 0 = player (bits 1..6 cleared: gather8 wants bit 4 clean)
                const uint32_t ox = o.x & 0x81818181u, oy = o.y & 0x81818181u;
                const uint32_t nx = ox >> 7, ny = oy >> 7;
                rows[ch] = (unsigned char)gather8<0>(~(ox | nx) & 0x01010101u, ~(oy | ny) & 0x01010101u);
                rows[rb + ch] = (unsigned char)gather8<0>(ox & ~nx, oy & ~ny);
            } else {
#pragma unroll
                for (int p = 0; p < NP; ++p)
                    if (p < P) {
                        const uint32_t pat = 0x01010101u * (uint32_t)p;
                        rows[p * rb + ch] = (unsigned char)gather8<0>(eq_bytes(o.x, pat), eq_bytes(o.y, pat));
                    }
            }
            // terrain in {0,1,2,3}: mountain = 01, structure (city / general) = 1x
            const uint32_t hx = t.x >> 1, hy = t.y >> 1;
            rows[R_MTN * rb + ch] = (unsigned char)gather8<0>(t.x & ~hx, t.y & ~hy);
            rows[R_STR * rb + ch] = (unsigned char)gather8<0>(hx, hy);
            rows[R_A2 * rb + ch] = (unsigned char)ge2_bits(a);
        }
        for (int ch = NC8 + ol; ch < NCH; ch += LPG) {  // bytes of the last word past the plane stride
            for (int p = 0; p < P; ++p) rows[p * rb + ch] = 0;
            rows[R_MTN * rb + ch] = 0xFF;
            rows[R_STR * rb + ch] = 0;
            rows[R_A2 * rb + ch] = 0;
        }
    };
    // word pass (octet): the four static "target is free" rows from the mountain row
    auto build_ok = [&](int lg) {
        const uint32_t *mtn = mrow(R_MTN, lg);
        auto freew = [&](int j) -> uint32_t { return ((unsigned)j < (unsigned)NW) ? (~mtn[j] & s_inb[j]) : 0u; };
        for (int j = ol; j < NW; j += LPG) {
            const uint32_t prev = freew(j - 1), cur = freew(j), next = freew(j + 1), in = s_inb[j];
            mrow(R_OK + 0, lg)[j] = __funnelshift_lc(prev, cur, W) & in;             // up:    c - W
            mrow(R_OK + 1, lg)[j] = __funnelshift_rc(cur, next, W) & in;             // down:  c + W
            mrow(R_OK + 2, lg)[j] = __funnelshift_l(prev, cur, 1) & s_nc0[j] & in;   // left:  c - 1
            mrow(R_OK + 3, lg)[j] = __funnelshift_r(cur, next, 1) & s_ncL[j] & in;   // right: c + 1
        }
    };
    // octet: scoreboard from the planes / bitboards (after a capture, a saturation, a reset; gen_observe)
    auto recount = [&](int lg, bool do_land, bool do_tot) {
        GameS &gs = s_game[lg];
        const int16_t *A = s_army + (size_t)lg * S;
        for (int p = 0; p < P; ++p) {
            int l = 0, sum = 0;
            for (int j = ol; j < NW; j += LPG) {
                uint32_t m = mrow(p, lg)[j] & s_inb[j];
                l += __popc(m);
                if (do_tot)
                    while (m) {
                        const int b = __ffs(m) - 1;
                        m &= m - 1;
                        sum += A[32 * j + b];
                    }
            }
#pragma unroll
            for (int o = LPG / 2; o >= 1; o >>= 1) {
                l += __shfl_xor_sync(gmask, l, o);
                sum += __shfl_xor_sync(gmask, sum, o);
            }
            if (ol == 0) {
                if (do_land) gs.land[p] = l;
                if (do_tot) gs.tot[p] = sum;
            }
        }
    };

    // ================================================================ prologue
    for (int t = tid; t < 34; t += blockDim.x) {
        const int j = t - 1;
        const bool in = j >= 0 && j < 32;
        s_nc0[j] = in ? kp.notcol0[j & 31] : 0u;
        s_ncL[j] = in ? kp.notcolL[j & 31] : 0u;
        s_inb[j] = in ? kp.inb[j & 31] : 0u;
    }
    pdl_launch_dependents();
    pdl_wait();
    const bool loading = !(flags & F_RESET) && nwg > 0;
    if (loading && lane == 0) {
        mbar_init(bar, 1);
        const uint32_t cells = (uint32_t)nwg * (uint32_t)S;
        mbar_expect_tx(bar, 4u * cells);
        bulk_g2s(smem_u32(s_army), B.army + (size_t)wg0 * S, 2u * cells, bar);
        bulk_g2s(smem_u32(s_owner), B.owner + (size_t)wg0 * S, cells, bar);
        bulk_g2s(smem_u32(s_terr), B.terrain + (size_t)wg0 * S, cells, bar);
    }
    if (loading && gvalid) {  // per-game scalars: every lane issues all loads (one round trip), then the octet scatters
        GameS &gs = s_game[sub];
        const size_t gp = (size_t)g * P + (size_t)min(ol, P - 1);
        const int32_t v_tot = __ldcg(B.army_total + gp), v_land = __ldcg(B.land + gp);
        const int32_t v_turn = __ldcg(B.turn + g);
        const uint32_t v_ep = __ldcg(B.episode + g), v_alive = __ldcg(B.alive + g), v_done = __ldcg(B.done + g);
        const int32_t v_win = __ldcg(B.winner + g);
        const unsigned long long v_dg = ((flags & F_DIGEST) && B.obs_digest) ? __ldcg(B.obs_digest + g) : 0ull;
        if (ol < P) { gs.tot[ol] = v_tot; gs.land[ol] = v_land; }
        if (ol == 0) { gs.turn = v_turn; gs.episode = v_ep; }
        if (ol == 1) { gs.alive = v_alive; gs.done = v_done; gs.winner = v_win; }
        if (ol == 2) {
            gs.flags = 0; gs.sat = 0; gs.dirtyO = 0; gs.dirtyA[0] = 0; gs.dirtyA[1] = 0; gs.rew_bits = 0;
            gs.digest = v_dg;
        }
    }
    __syncthreads();  // the only CTA barrier: tables (and the mbarrier init) are visible
    if (nwg <= 0) return;

    if (flags & F_RESET) {
        if (gvalid && ol == 0) {
            GameS &gs = s_game[sub];
            gs.episode = (flags & F_KEEP_EPISODE) ? B.episode[g] : 0u;
            gs.flags = 0; gs.done = 0; gs.winner = -1; gs.digest = 0; gs.sat = 0;
            gs.dirtyO = 0; gs.dirtyA[0] = 0; gs.dirtyA[1] = 0; gs.rew_bits = 0;
            B.episode[g] = gs.episode;
            B.episodes_done[g] = 0; B.truncations[g] = 0; B.sat_events[g] = 0;
            if (B.invalid_actions) B.invalid_actions[g] = 0;
            for (int p = 0; p < P; ++p) B.wins[(size_t)g * P + p] = 0;
        }
        __syncwarp();
        for (int lg = 0; lg < nwg; ++lg) generate(lg);
    } else {
        mbar_wait(bar, 0);
    }
    if ((flags & F_OBSERVE_ONLY) && gvalid) {
        // R40: gen_observe takes a state written by the caller.  In every state the rules produce, the GENERAL cells
        // are exactly the cells general_cell[p] of their owners (both generators place them so; a captured general
        // becomes a CITY, R11).  A GENERAL cell that is nobody's recorded general -- an "unclaimed general", a second
        // one -- is turned into a CITY here, so that no rule ever meets one (the two step kernels tell a general by
        // the terrain and by general_cell respectively; on well-formed states these agree).
        int8_t *Tr = s_terr + (size_t)sub * S;
        const int8_t *O = s_owner + (size_t)sub * S;
        bool fixed = false;
        for (int c = ol; c < HW; c += LPG)
            if (Tr[c] == T_GENERAL) {
                const int o = O[c];
                if (o < 0 || o >= P || B.general_cell[(size_t)g * P + o] != c) { Tr[c] = (int8_t)T_CITY; fixed = true; }
            }
        if (fixed) atomicOr(&s_game[sub].flags, (uint32_t)GF_TERRAIN_DIRTY);
    }
    __syncwarp();
    if (gvalid) build_game(sub);
    __syncwarp();
    if (gvalid) {
        build_ok(sub);
        if (flags & F_OBSERVE_ONLY) recount(sub, true, true);
    }
    __syncwarp();

    // ---------------------------------------------------------------- a12: valid-action sampler (R24, R25)
    // All players of a game are drawn in one instruction stream: the LPP lanes (pl, 0..LPP-1) of the octet
    // serve player pl and split the NW bitboard words among themselves (WS consecutive words each).  The valid
    // list is ordered (direction, cell).  Returns player pl's action on every lane serving pl.  No lane leaves
    // early, so the octet stays converged for the shuffles.
    auto sample = [&](int lg, uint32_t gstep) -> int {
        const int p = min(pl, P - 1);  // lanes past the last player shadow it (their result is ignored)
        const uint32_t gid = kp.gid_base + (uint32_t)(wg0 + lg);
        uint32_t w[4];
        philox(0u, gid, gstep, (DOM_ACTION << 24) | (uint32_t)p, kp.key0, kp.key1, w);
        const uint32_t *own = mrow(p, lg), *a2 = mrow(R_A2, lg), *ok = mrow(R_OK, lg);
        const int js = sl * WS, je = min(js + WS, NW);
        // count pass: my words' valid moves per direction, packed 2 x 16 bits
        uint32_t ln01 = 0, ln23 = 0;
        for (int j = js; j < je; ++j) {
            const uint32_t src = own[j] & a2[j];
            ln01 += (uint32_t)__popc(src & ok[j]) | ((uint32_t)__popc(src & ok[RW + j]) << 16);
            ln23 += (uint32_t)__popc(src & ok[2 * RW + j]) | ((uint32_t)__popc(src & ok[3 * RW + j]) << 16);
        }
        uint32_t n01 = ln01, n23 = ln23;
#pragma unroll
        for (int o = LPP / 2; o >= 1; o >>= 1) {
            n01 += __shfl_xor_sync(gmask, n01, o);
            n23 += __shfl_xor_sync(gmask, n23, o);
        }
        const uint32_t n0 = n01 & 0xFFFFu, n1 = n01 >> 16, n2 = n23 & 0xFFFFu, n3 = n23 >> 16;
        const uint32_t total = n0 + n1 + n2 + n3;
        const int half = (w[2] < kp.half_thr) ? 1 : 0;
        int action = 0;
        bool decided = (w[0] < kp.pass_thr) || total == 0;
        if (kp.bias_thr) {  // uniform: config 4's policy
            // largest owned stack, ties -> lowest cell index: max of (army + 1) << 10 | (1023 - cell)
            const int16_t *A = s_army + (size_t)lg * S;
            uint32_t best = 0;
            for (int j = js; j < je; ++j) {
                uint32_t m = own[j] & s_inb[j];
                while (m) {
                    const int c = 32 * j + __ffs(m) - 1;
                    m &= m - 1;
                    best = max(best, (((uint32_t)A[c] + 1u) << 10) | (uint32_t)(1023 - c));
                }
            }
#pragma unroll
            for (int o = LPP / 2; o >= 1; o >>= 1) best = max(best, __shfl_xor_sync(gmask, best, o));
            if (!decided && w[3] < kp.bias_thr && best) {
                const int bc = 1023 - (int)(best & 1023u), jb = bc >> 5;
                const uint32_t src = (own[jb] & a2[jb]) >> (bc & 31);
                uint32_t vb = 0;
#pragma unroll
                for (int d = 0; d < 4; ++d) vb |= ((src & (ok[d * RW + jb] >> (bc & 31))) & 1u) << d;
                if (vb) {
                    const int d = nth_bit(vb, mulhi32(w[1], (uint32_t)__popc(vb)));
                    action = bc * 9 + 1 + 2 * d + half;
                    decided = true;
                }
            }
        }
        uint32_t idx = mulhi32(w[1], total);
        int d = 0;
        uint32_t cnt = ln01 & 0xFFFFu;
        if (idx >= n0) { idx -= n0; d = 1; cnt = ln01 >> 16;
            if (idx >= n1) { idx -= n1; d = 2; cnt = ln23 & 0xFFFFu;
                if (idx >= n2) { idx -= n2; d = 3; cnt = ln23 >> 16; } } }
        uint32_t incl = cnt;
#pragma unroll
        for (int o = 1; o < LPP; o <<= 1) {
            const uint32_t t = __shfl_up_sync(gmask, incl, o, LPP);
            if (sl >= o) incl += t;
        }
        int cell = -1;
        if (!decided && idx < incl && idx >= incl - cnt) {  // the idx-th move of direction d starts in my words
            uint32_t r = idx - (incl - cnt), vw = 0;
            int j = js;
            for (; j < je; ++j) {
                vw = own[j] & a2[j] & ok[d * RW + j];
                const uint32_t c = (uint32_t)__popc(vw);
                if (r < c) break;
                r -= c;
            }
            cell = 32 * j + nth_bit(vw, r);
        }
        const int leader = (int)(lane & ~(uint32_t)(LPP - 1));
        const uint32_t mine = (__ballot_sync(gmask, cell >= 0) >> leader) & ((1u << LPP) - 1u);
        cell = __shfl_sync(gmask, cell, mine ? leader + __ffs(mine) - 1 : (int)lane);
        if (mine) action = cell * 9 + 1 + 2 * d + half;
        return action;
    };

    // ---------------------------------------------------------------- a2-a5: moves of one game, one lane
    auto set_bit = [&](uint32_t *row, int c, bool on) {
        const uint32_t bit = 1u << (c & 31);
        if (on) row[c >> 5] |= bit; else row[c >> 5] &= ~bit;
    };

    auto play_moves = [&](int lg) {
        GameS &gs = s_game[lg];
        int16_t *A = s_army + (size_t)lg * S;
        int8_t *O = s_owner + (size_t)lg * S, *Tr = s_terr + (size_t)lg * S;
        uint32_t *a2row = mrow(R_A2, lg);
        const int gg = wg0 + lg;
        const int first = (kp.rule_flags & GEN_RULE_ROTATE_PRIORITY) ? (gs.turn % P) : 0;
        uint32_t dA0 = 0, dA1 = 0, dO = 0, gflags = 0;
        int bad = 0;  // non-pass actions that are not applied (diagnostic counter invalid_actions)
        for (int i = 0; i < P; ++i) {
            int p = first + i;
            if (p >= P) p -= P;
            const int a = gs.act[p];
            if (a == 0) continue;
            if (a < 0 || a >= 9 * HW) { ++bad; continue; }
            const int cell = (int)(((uint32_t)a * 7282u) >> 16);  // a / 9 for a < 9 * 1024
            const int kk = a - 9 * cell;
            if (kk == 0) continue;
            const int dir = (kk - 1) >> 1, half = (kk - 1) & 1;
            const int r = row_of(cell), col = cell - r * W;
            int dst;
            bool ok;
            if (dir == 0) { dst = cell - W; ok = r > 0; }
            else if (dir == 1) { dst = cell + W; ok = r < H - 1; }
            else if (dir == 2) { dst = cell - 1; ok = col > 0; }
            else { dst = cell + 1; ok = col < W - 1; }
            if (!ok) { ++bad; continue; }
            const int asrc = A[cell];
            if (O[cell] != p || asrc < 2 || Tr[dst] == T_MOUNTAIN) { ++bad; continue; }
            const int m = half ? (asrc >> 1) : (asrc - 1);  // R4
            const int nsrc = asrc - m;
            const int t = O[dst], d = A[dst];
            const bool dst_general = Tr[dst] == T_GENERAL;
            int ndst, nown = t;
            bool captured = false;
            const bool ally = teams && t >= 0 && t != p && ((team_mask(p) >> t) & 1u);
            if (t == p || ally) {  // R8 / P:L97, R19
                ndst = d + m;
                if (ndst > 32767) { ndst = 32767; gs.sat += 1; gflags |= GF_RECOUNT; }
                if (ally) {
                    if (!dst_general) { nown = p; gs.tot[p] += d; gs.tot[t] -= d; }
                    else { gs.tot[p] -= m; gs.tot[t] += m; }
                }
            } else if (m > d) {
                ndst = m - d;
                nown = p;
                captured = dst_general && t >= 0;  // R11, R12
                gs.tot[p] -= d;
                if (t >= 0) gs.tot[t] -= d;
            } else {
                ndst = d - m;  // tie -> 0, previous owner keeps the cell
                gs.tot[p] -= m;
                if (t >= 0) gs.tot[t] -= m;
            }
            A[cell] = (int16_t)nsrc;
            A[dst] = (int16_t)ndst;
            if (cell < 512) dA0 |= 1u << (cell >> 4); else dA1 |= 1u << ((cell >> 4) & 31);
            if (dst < 512) dA0 |= 1u << (dst >> 4); else dA1 |= 1u << ((dst >> 4) & 31);
            set_bit(a2row, cell, nsrc >= 2);
            set_bit(a2row, dst, ndst >= 2);
            if (nown != t) {
                O[dst] = (int8_t)nown;
                dO |= 1u << (dst >> 5);
                set_bit(mrow(nown, lg), dst, true);
                gs.land[nown] += 1;
                if (t >= 0) { set_bit(mrow(t, lg), dst, false); gs.land[t] -= 1; }
            }
            if (captured) {  // a4: land transfer (R11)
                const int q = t;
                Tr[dst] = (int8_t)T_CITY;
                gs.alive &= ~(1u << q);
                B.general_cell[(size_t)gg * P + q] = -1;
                const bool fl = (kp.rule_flags & GEN_RULE_CAPTURE_HALF_FLOOR) != 0;
                uint32_t *oq = mrow(q, lg), *op = mrow(p, lg);
                for (int j = 0; j < NW; ++j) {
                    uint32_t wq = oq[j];
                    op[j] |= wq;
                    oq[j] = 0;
                    while (wq) {
                        const int c = 32 * j + __ffs(wq) - 1;
                        wq &= wq - 1;
                        O[c] = (int8_t)p;
                        const int av = A[c];
                        A[c] = (int16_t)(fl ? (av >> 1) : ((av + 1) >> 1));
                    }
                }
                gflags |= GF_REBUILD | GF_RECOUNT | GF_TERRAIN_DIRTY | GF_ALL_DIRTY;
            }
        }
        // a6: turn counter; growth itself is applied by the next parallel pass (R1, R2, R3)
        if (bad && B.invalid_actions) B.invalid_actions[gg] += (uint32_t)bad;
        const int turn = gs.turn + 1;
        gs.turn = turn;
        if ((turn & 1) == 0) gflags |= GF_GROW_EVEN;
        if (turn % 50 == 0) gflags |= GF_GROW_TICK;
        if (gflags) gs.flags |= gflags;
        if (dA0) gs.dirtyA[0] |= dA0;
        if (dA1) gs.dirtyA[1] |= dA1;
        if (dO) gs.dirtyO |= dO;
    };

    // ---------------------------------------------------------------- a6: growth
    // tick turns (every 50th): cell pass over one chunk, +1 on owned cells (+2 on owned structures)
    auto grow_chunk = [&](int lg, int ch, uint32_t gflags) {
        GameS &gs = s_game[lg];
        const uint32_t sb = mrow8(R_STR, lg)[ch];
        uint32_t ownedb = 0;
        for (int p = 0; p < P; ++p) ownedb |= mrow8(p, lg)[ch];
        const uint32_t e = (gflags & GF_GROW_EVEN) ? (sb & ownedb) : 0u;
        const uint32_t t = (gflags & GF_GROW_TICK)
                               ? ((kp.rule_flags & GEN_RULE_TICK_PLAIN_ONLY) ? (ownedb & ~sb) : ownedb) : 0u;
        if ((e | t) == 0) return;
        uint4 *ap = reinterpret_cast<uint4 *>(s_army + (size_t)lg * S + 8 * ch);
        uint4 a = *ap;
        uint32_t aw[4] = {a.x, a.y, a.z, a.w};
        bool sat = false;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const uint32_t lo = ((e >> (2 * k)) & 1u) + ((t >> (2 * k)) & 1u);
            const uint32_t hi = ((e >> (2 * k + 1)) & 1u) + ((t >> (2 * k + 1)) & 1u);
            aw[k] += lo | (hi << 16);
            sat |= (aw[k] & 0x80008000u) != 0;
        }
        if (sat) {  // R21: every +1 that would pass 32767 is one saturation event
            int ev = 0;
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                uint32_t lo = aw[k] & 0xFFFFu, hi = aw[k] >> 16;
                if (lo > 32767u) { ev += (int)(lo - 32767u); lo = 32767u; }
                if (hi > 32767u) { ev += (int)(hi - 32767u); hi = 32767u; }
                aw[k] = lo | (hi << 16);
            }
            atomicAdd(&gs.sat, (uint32_t)ev);
            atomicOr(&gs.flags, GF_RECOUNT);
        }
        a.x = aw[0]; a.y = aw[1]; a.z = aw[2]; a.w = aw[3];
        *ap = a;
        mrow8(R_A2, lg)[ch] = (unsigned char)ge2_bits(a);
        atomicOr(&gs.dirtyA[ch >> 6], 1u << ((ch >> 1) & 31));
        for (int p = 0; p < P; ++p) {
            const uint32_t ob = mrow8(p, lg)[ch];
            const int inc = __popc(e & ob) + __popc(t & ob);
            if (inc) atomicAdd(&gs.tot[p], inc);
        }
    };
    // even turns that are no tick: +1 on the few owned structures, found by bit iteration (octet)
    auto grow_structures = [&](int lg) {
        GameS &gs = s_game[lg];
        int16_t *A = s_army + (size_t)lg * S;
        uint32_t dA0 = 0, dA1 = 0;
        for (int j = ol; j < NW; j += LPG) {
            const uint32_t sw = mrow(R_STR, lg)[j];
            if (sw == 0) continue;
            uint32_t a2w = mrow(R_A2, lg)[j];
            bool changed = false;
            for (int p = 0; p < P; ++p) {
                uint32_t m = sw & mrow(p, lg)[j];
                if (m == 0) continue;
                int inc = 0;
                while (m) {
                    const int b = __ffs(m) - 1;
                    m &= m - 1;
                    const int c = 32 * j + b, av = A[c];
                    if (av >= 32767) { atomicAdd(&gs.sat, 1u); continue; }  // R21
                    A[c] = (int16_t)(av + 1);
                    inc += 1;
                    if (av == 1) { a2w |= 1u << b; changed = true; }
                    if (c < 512) dA0 |= 1u << (c >> 4); else dA1 |= 1u << ((c >> 4) & 31);
                }
                if (inc) atomicAdd(&gs.tot[p], inc);
            }
            if (changed) mrow(R_A2, lg)[j] = a2w;
        }
        if (dA0) atomicOr(&gs.dirtyA[0], dA0);
        if (dA1) atomicOr(&gs.dirtyA[1], dA1);
    };

    // ---------------------------------------------------------------- a7-a9: end of turn, one lane per game
    auto write_result = [&](size_t slot, int gg, int rew_bits, uint32_t done, int winner) {
        int8_t *rw = B.reward + (slot * kp.N + gg) * P;
        if (rew_bits == 0x5555 >> (16 - 2 * P) && (P == 2 || P == 4 || P == 8)) {  // all zero: one store
            if (P == 2) *reinterpret_cast<uint16_t *>(rw) = 0;
            else if (P == 4) *reinterpret_cast<uint32_t *>(rw) = 0;
            else *reinterpret_cast<uint2 *>(rw) = make_uint2(0u, 0u);
        } else {
            for (int p = 0; p < P; ++p) rw[p] = (int8_t)(((rew_bits >> (2 * p)) & 3) - 1);
        }
        B.done[slot * kp.N + gg] = (uint8_t)done;
        B.winner[slot * kp.N + gg] = (int8_t)winner;
    };
    auto finish_turn = [&](int lg, size_t slot, bool write_out) {
        GameS &gs = s_game[lg];
        const int gg = wg0 + lg;
        if (gs.sat) { B.sat_events[gg] += gs.sat; gs.sat = 0; }
        const int zero_bits = 0x5555 >> (16 - 2 * P);
        const bool truncated_now = kp.max_turns > 0 && gs.turn >= kp.max_turns;
        if (gs.alive == allp && !truncated_now && kp.n_teams > 1) {  // the common case: nothing ends
            gs.done = 0;
            gs.winner = -1;
            gs.rew_bits = zero_bits;
            if (write_out) write_result(slot, gg, zero_bits, 0u, -1);
            return;
        }
        int living = 0, last = -1;
        for (int t = 0; t < kp.n_teams; ++t) {
            const uint32_t tm = (((1u << kp.team_size) - 1u) << (t * kp.team_size)) & allp;
            if (gs.alive & tm) { ++living; last = t; }
        }
        const bool terminated = living <= 1;
        const bool truncated = !terminated && truncated_now;
        gs.done = (terminated ? 1u : 0u) | (truncated ? 2u : 0u);
        gs.winner = terminated ? last : -1;
        int rew_bits = 0;
        for (int p = 0; p < P; ++p) {
            const int r = terminated ? ((p / kp.team_size == last) ? 1 : -1) : 0;
            rew_bits |= (r + 1) << (2 * p);
            if (r > 0) B.wins[(size_t)gg * P + p] += 1;
        }
        gs.rew_bits = rew_bits;
        if (write_out) write_result(slot, gg, rew_bits, gs.done, gs.winner);
        if (gs.done) {
            B.episodes_done[gg] += 1;
            if (truncated) B.truncations[gg] += 1;
            if (kp.auto_reset) {  // a9 (R17): reward / done describe the finished episode, state + obs the new one
                gs.episode += 1;
                B.episode[gg] = gs.episode;
                gs.flags |= GF_RESET;
            }
        }
    };

    // ---------------------------------------------------------------- a10: fog of war (all players at once)
    // vis = 3x3 dilation of the team's cells.  Sub-lane (pl, sl) streams through its WS words of player pl's
    // row with a sliding window: tw = team-owned words, h = horizontally dilated words, both in registers.
    auto compute_vis = [&](int lg) {
        if (pl >= P) return;
        const int js = sl * WS, je = min(js + WS, NW);
        if (js >= je) return;
        uint32_t *vr = mrow(R_VIS + pl, lg);
        const uint32_t *own = mrow(pl, lg);
        const uint32_t members = teams ? team_mask(pl) : 0u;
        auto tw = [&](int j) -> uint32_t {
            if ((unsigned)j >= (unsigned)NW) return 0u;
            if (!teams) return own[j];
            uint32_t tm = 0;
            for (int q = 0; q < P; ++q)
                if ((members >> q) & 1u) tm |= mrow(q, lg)[j];
            return tm;
        };
        auto hdil = [&](uint32_t a, uint32_t b, uint32_t c, int j) -> uint32_t {  // s_nc0 / s_ncL are 0 off the board
            return b | (__funnelshift_l(a, b, 1) & s_nc0[j]) | (__funnelshift_r(b, c, 1) & s_ncL[j]);
        };
        uint32_t t1 = tw(js - 1), t2 = tw(js), t3 = tw(js + 1);
        uint32_t hm = hdil(tw(js - 2), t1, t2, js - 1), hc = hdil(t1, t2, t3, js);
        for (int j = js; j < je; ++j) {
            const uint32_t t4 = tw(j + 2);
            const uint32_t hn = hdil(t2, t3, t4, j + 1);
            vr[j] = (hc | __funnelshift_lc(hm, hc, W) | __funnelshift_rc(hc, hn, W)) & s_inb[j];
            hm = hc; hc = hn; t2 = t3; t3 = t4;
        }
    };

    // ---------------------------------------------------------------- a11: observation planes (octet)
    // per player, per 8-cell chunk: one 16-byte and three 8-byte streaming stores; the 8 lanes of the octet
    // write 128 / 64 contiguous bytes per instruction (full 32-byte sectors)
    auto emit_planes = [&](int lg, size_t slot) {
        const size_t base = (slot * (size_t)kp.N + (size_t)(wg0 + lg)) * (size_t)P * (size_t)S;
        const unsigned char *sa = reinterpret_cast<const unsigned char *>(s_army + (size_t)lg * S) + 16 * ol;
        const unsigned char *so = reinterpret_cast<const unsigned char *>(s_owner + (size_t)lg * S) + 8 * ol;
        const unsigned char *st = reinterpret_cast<const unsigned char *>(s_terr + (size_t)lg * S) + 8 * ol;
        const int nit = (NC8 - ol + LPG - 1) / LPG;  // chunks of this lane: ol, ol + 8, ...
        for (int p = 0; p < P; ++p) {
            const unsigned char *sv = mrow8(R_VIS + p, lg) + ol;
            unsigned char *ga = reinterpret_cast<unsigned char *>(B.obs_army + base + (size_t)p * S) + 16 * ol;
            unsigned char *go = reinterpret_cast<unsigned char *>(B.obs_owner + base + (size_t)p * S) + 8 * ol;
            unsigned char *gt = reinterpret_cast<unsigned char *>(B.obs_terrain + base + (size_t)p * S) + 8 * ol;
            unsigned char *gv = reinterpret_cast<unsigned char *>(B.obs_vis + base + (size_t)p * S) + 8 * ol;
            unsigned char *gp = reinterpret_cast<unsigned char *>(B.obs_packed + base + (size_t)p * S) + 8 * ol;
#pragma unroll 3
            for (int i = 0; i < nit; ++i) {
                const uint4 a = *reinterpret_cast<const uint4 *>(sa + 128 * i);
                const uint2 o = *reinterpret_cast<const uint2 *>(so + 64 * i);
                const uint2 t = *reinterpret_cast<const uint2 *>(st + 64 * i);
                const uint32_t vb = sv[8 * i];
                const uint32_t s0 = nib_sign(vb & 15u), s1 = nib_sign(vb >> 4);
                const uint32_t m0 = prmt(s0, 0u, 0xBA98u), m1 = prmt(s1, 0u, 0xBA98u);
                uint4 oa;
                oa.x = a.x & prmt(s0, 0u, 0x9988u); oa.y = a.y & prmt(s0, 0u, 0xBBAAu);
                oa.z = a.z & prmt(s1, 0u, 0x9988u); oa.w = a.w & prmt(s1, 0u, 0xBBAAu);
                __stcs(reinterpret_cast<uint4 *>(ga + 128 * i), oa);
                if (B.obs_packed) {  // R33: 0x80 | terrain << 4 | (owner + 2) under the fog mask
                    const uint32_t qx = 0x80808080u | ((t.x << 4) & 0x30303030u) |
                                        (((o.x & 0x0F0F0F0Fu) + 0x02020202u) & 0x0F0F0F0Fu);
                    const uint32_t qy = 0x80808080u | ((t.y << 4) & 0x30303030u) |
                                        (((o.y & 0x0F0F0F0Fu) + 0x02020202u) & 0x0F0F0F0Fu);
                    __stcs(reinterpret_cast<uint2 *>(gp + 64 * i), make_uint2(qx & m0, qy & m1));
                    continue;
                }
                uint2 oo, ot, ov;
                oo.x = (o.x & m0) | (~m0 & 0xFEFEFEFEu); oo.y = (o.y & m1) | (~m1 & 0xFEFEFEFEu);
                ot.x = (t.x & m0) | (~m0 & 0x04040404u); ot.y = (t.y & m1) | (~m1 & 0x04040404u);
                ov.x = m0 & 0x01010101u; ov.y = m1 & 0x01010101u;
                __stcs(reinterpret_cast<uint2 *>(go + 64 * i), oo);
                __stcs(reinterpret_cast<uint2 *>(gt + 64 * i), ot);
                __stcs(reinterpret_cast<uint2 *>(gv + 64 * i), ov);
            }
        }
    };

    // R28: h_p = sum_c pack(p, c) * key(c), pack = army | (owner + 2) << 16 | terrain << 20 | vis << 24.
    // A fogged cell packs to 0x400000, a visible one to x | 0x1000000, so
    // pack - 0x400000 = vis ? (x | 0xC00000) : 0 (terrain <= 3 leaves bits 22, 23 clear) and
    // h_p = 0x400000 * sum(key) + sum_c vis & (x | 0xC00000) * key(c).  All 8 lanes of the octet call this.
    // Instruction diet (this loop was half of the fused rollout's instruction stream): x = army | ob << 16 | 0xC00000
    // is ONE byte permute per cell (the 0xC0 rides on the ob byte, the top byte is the sign replica of the army's
    // high byte, which is 0 since army <= 32767); x * key mod 2^64 is accumulated per player as a 64-bit sum of
    // x * key_lo (one wide multiply-add) and a 32-bit sum of x * key_hi (one multiply-add) of x-or-0 by the player's
    // fog bit -- no 64-bit product is formed and then added under a predicate twice (inline PTX: the compiler
    // turns every other spelling back into that).
    auto chain_digest = [&](int lg, bool active) {
        uint64_t h[NP];
#pragma unroll
        for (int p = 0; p < NP; ++p) h[p] = 0;
        if (active) {
            uint64_t lo[NP];
            uint32_t hi[NP];
#pragma unroll
            for (int p = 0; p < NP; ++p) { lo[p] = 0; hi[p] = 0; }
            for (int ch = ol; ch < NC8; ch += LPG) {
                uint32_t vb[NP], any = 0;
#pragma unroll
                for (int p = 0; p < NP; ++p) { vb[p] = (p < P) ? mrow8(R_VIS + p, lg)[ch] : 0u; any |= vb[p]; }
                if (any == 0) continue;
                const uint4 a = *reinterpret_cast<const uint4 *>(s_army + (size_t)lg * S + 8 * ch);
                const uint2 o = *reinterpret_cast<const uint2 *>(s_owner + (size_t)lg * S + 8 * ch);
                const uint2 t = *reinterpret_cast<const uint2 *>(s_terr + (size_t)lg * S + 8 * ch);
                // per byte: (owner + 2) | terrain << 4 | 0xC0
                const uint32_t otx = (((o.x & 0x0F0F0F0Fu) + 0x02020202u) & 0x0F0F0F0Fu) | (t.x << 4) | 0xC0C0C0C0u;
                const uint32_t oty = (((o.y & 0x0F0F0F0Fu) + 0x02020202u) & 0x0F0F0F0Fu) | (t.y << 4) | 0xC0C0C0C0u;
                const uint32_t aw[4] = {a.x, a.y, a.z, a.w};
                // the eight keys of the chunk: four 16-byte loads (cells past the board are never visible)
                unsigned long long key[8];
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    const ulonglong2 kk = __ldg(reinterpret_cast<const ulonglong2 *>(g_digest_keys.k + 8 * ch) + i);
                    key[2 * i] = kk.x; key[2 * i + 1] = kk.y;
                }
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    // bytes of x: army low, army high, ob | 0xC0, 0 (sign replica of the army's high byte)
                    const uint32_t sel = (i & 1) ? (0xB032u | ((4u + (i & 3)) << 8)) : (0x9010u | ((4u + (i & 3)) << 8));
                    const uint32_t x = prmt(aw[i >> 1], (i < 4) ? otx : oty, sel);
                    const uint32_t klo = (uint32_t)key[i], khi = (uint32_t)(key[i] >> 32);
#pragma unroll
                    for (int p = 0; p < NP; ++p)
                        if (p < P)  // four instructions per cell and player: fog bit -> x or 0, two multiply-adds
                            asm("{\n\t.reg .pred q;\n\t.reg .b32 t, xm;\n\t"
                                "and.b32 t, %2, %3;\n\t"
                                "setp.ne.u32 q, t, 0;\n\t"
                                "selp.b32 xm, %4, 0, q;\n\t"
                                "mad.wide.u32 %0, xm, %5, %0;\n\t"
                                "mad.lo.u32 %1, xm, %6, %1;\n\t}"
                                : "+l"(lo[p]), "+r"(hi[p])
                                : "r"(vb[p]), "r"(1u << i), "r"(x), "r"(klo), "r"(khi));
                }
            }
#pragma unroll
            for (int p = 0; p < NP; ++p) h[p] = lo[p] + ((uint64_t)hi[p] << 32);
        }
#pragma unroll
        for (int p = 0; p < NP; ++p) {
#pragma unroll
            for (int o = LPG / 2; o >= 1; o >>= 1) h[p] += __shfl_xor_sync(FULL, h[p], o);
        }
        if (active && ol == 0) {
            GameS &gs = s_game[lg];
            const uint64_t c0 = 0x400000ull * kp.key_sum;
            uint64_t dg = gs.digest;
#pragma unroll
            for (int p = 0; p < NP; ++p)
                if (p < P) dg = mix64(dg ^ (c0 + h[p]));
            const uint64_t tail = (uint64_t)gs.done | ((uint64_t)(uint8_t)(gs.winner + 2) << 8) |
                                  ((uint64_t)(uint32_t)gs.rew_bits << 16);
            gs.digest = mix64(dg ^ tail);
        }
    };

    if (flags & F_SAMPLE_ONLY) {
        if (gvalid) {
            const GameS &gs = s_game[sub];
            const bool frozen = !kp.auto_reset && gs.done != 0;
            const int a = frozen ? 0 : sample(sub, kp.global_step0);
            if (sl == 0 && pl < P) kp.sample_out[(size_t)g * P + pl] = a;
        }
        return;
    }

    // ================================================================ K turns
    const bool every = (flags & F_OBS_EVERY) != 0;
    for (int k = 0; k < K; ++k) {
        const size_t slot = every ? (size_t)k : 0;
        const uint32_t gstep = kp.global_step0 + (uint32_t)k;
        const bool last_step = (k == K - 1);
        // ---- actions (all players at once), then the moves (lane 0 of the octet)
        bool frozen = false;
        if (gvalid) {
            GameS &gs = s_game[sub];
            frozen = !kp.auto_reset && gs.done != 0;  // R31
            int a = 0;
            if (!frozen) {
                if (flags & F_SAMPLER) a = sample(sub, gstep);
                else if (sl == 0 && pl < P) a = kp.actions[(size_t)g * P + pl];
            }
            if (sl == 0 && pl < P) {
                gs.act[pl] = a;
                if (B.actions_out) B.actions_out[(slot * kp.N + g) * P + pl] = a;
            }
        }
        __syncwarp();
        if (gvalid && ol == 0) {
            if (frozen) s_game[sub].flags |= GF_FROZEN;
            else play_moves(sub);
        }
        __syncwarp();
        // ---- parallel pass: rebuild after a capture, growth, recount after a saturation
        if (gvalid) {
            GameS &gs = s_game[sub];
            const uint32_t gf = gs.flags;
            if (gf & (GF_GROW_EVEN | GF_GROW_TICK | GF_REBUILD | GF_RECOUNT)) {
                if (gf & GF_REBUILD) {
                    build_game(sub);
                    __syncwarp(gmask);
                    recount(sub, true, false);
                }
                if (gf & GF_GROW_TICK) {
                    for (int ch = ol; ch < NC8; ch += LPG) grow_chunk(sub, ch, gf);
                } else if (gf & GF_GROW_EVEN) {
                    grow_structures(sub);
                }
                __syncwarp(gmask);
                if (gs.flags & GF_RECOUNT) recount(sub, false, true);
                __syncwarp(gmask);
                if (ol == 0) gs.flags &= ~(GF_GROW_EVEN | GF_GROW_TICK | GF_REBUILD | GF_RECOUNT);
            }
        }
        __syncwarp();
        // ---- end of turn
        bool want_reset = false;
        if (gvalid && ol == 0) {
            GameS &gs = s_game[sub];
            if (frozen) {
                gs.rew_bits = 0x5555 >> (16 - 2 * P);
                if (every || last_step) write_result(slot, g, gs.rew_bits, gs.done, gs.winner);
            } else {
                finish_turn(sub, slot, every || last_step);
            }
            want_reset = (gs.flags & GF_RESET) != 0;
        }
        const uint32_t rs = __ballot_sync(FULL, want_reset);  // bit sub * LPG: game sub must be regenerated
        if (rs) {
            for (int lg = 0; lg < nwg; ++lg)
                if ((rs >> (lg * LPG)) & 1u) generate(lg);
            const bool mine = gvalid && ((rs >> (sub * LPG)) & 1u);
            if (mine) build_game(sub);
            __syncwarp();
            if (mine) {
                build_ok(sub);
                if (ol == 0) s_game[sub].flags &= ~GF_RESET;
            }
        }
        __syncwarp();
        // ---- R34: slot (turn mod 512) of the scoreboard history ring, the scoreboard as this turn leaves it
        if (B.score_hist && gvalid && !frozen && ol < P) {
            const GameS &gs = s_game[sub];
            *reinterpret_cast<int2 *>(B.score_hist + (((size_t)g * 512 + (size_t)(gs.turn & 511)) * P + ol) * 2) =
                make_int2(gs.land[ol], gs.tot[ol]);
        }
        // ---- a10 + a11 (R32: the state at the end of the call)
        const bool planes = (flags & F_OBS_PLANES) && (every || last_step);
        if (planes || (flags & F_DIGEST)) {
            if (gvalid) compute_vis(sub);
            __syncwarp();
            if (planes && gvalid) emit_planes(sub, slot);
            if (flags & F_DIGEST) chain_digest(sub, gvalid && !frozen);
        }
    }

    if (K == 0) {  // gen_reset / gen_observe: observation of the state as it stands
        if (gvalid) {
            if ((flags & F_RESET) && B.score_hist && ol < P) {  // R34: turn 0 of the ring
                const GameS &gs = s_game[sub];
                *reinterpret_cast<int2 *>(B.score_hist + (((size_t)g * 512) * P + ol) * 2) = make_int2(gs.land[ol], gs.tot[ol]);
            }
            compute_vis(sub);
            if ((flags & F_RESET) && ol == 0) {
                GameS &gs = s_game[sub];
                gs.rew_bits = 0x5555 >> (16 - 2 * P);
                write_result(0, g, gs.rew_bits, 0u, -1);
            }
        }
        __syncwarp();
        if ((flags & F_OBS_PLANES) && gvalid) emit_planes(sub, 0);
        if ((flags & F_RESET) && (flags & F_DIGEST)) chain_digest(sub, gvalid);
    }

    // ================================================================ store state
    __syncwarp();
    if (gvalid) {
        const GameS &gs = s_game[sub];
        const size_t gbase = (size_t)g * S;
        const uint32_t gf = gs.flags;
        if (gf & GF_ALL_DIRTY) {
            for (int u = ol; u < S / 8; u += LPG)
                *reinterpret_cast<uint4 *>(B.army + gbase + 8 * u) =
                    *reinterpret_cast<const uint4 *>(s_army + (size_t)sub * S + 8 * u);
            for (int u = ol; u < S / 16; u += LPG)
                *reinterpret_cast<uint4 *>(B.owner + gbase + 16 * u) =
                    *reinterpret_cast<const uint4 *>(s_owner + (size_t)sub * S + 16 * u);
        } else {
            // dirty 32-byte sectors of the army plane (16 cells): lane l takes the sectors u = l (mod 8)
#pragma unroll
            for (int hw = 0; hw < 2; ++hw) {
                uint32_t m = gs.dirtyA[hw] & (0x01010101u << ol);
                while (m) {
                    const int u = 32 * hw + __ffs(m) - 1;
                    m &= m - 1;
                    const uint4 *src = reinterpret_cast<const uint4 *>(s_army + (size_t)sub * S + 16 * u);
                    uint4 *dst = reinterpret_cast<uint4 *>(B.army + gbase + 16 * u);
                    dst[0] = src[0];
                    dst[1] = src[1];
                }
            }
            // dirty 32-cell groups of the owner plane
            uint32_t m = gs.dirtyO & (0x01010101u << ol);
            while (m) {
                const int u = __ffs(m) - 1;
                m &= m - 1;
                const uint4 *src = reinterpret_cast<const uint4 *>(s_owner + (size_t)sub * S + 32 * u);
                uint4 *dst = reinterpret_cast<uint4 *>(B.owner + gbase + 32 * u);
                dst[0] = src[0];
                if (32 * u + 16 < S) dst[1] = src[1];
            }
        }
        if (gf & GF_TERRAIN_DIRTY)
            for (int u = ol; u < S / 16; u += LPG)
                *reinterpret_cast<uint4 *>(B.terrain + gbase + 16 * u) =
                    *reinterpret_cast<const uint4 *>(s_terr + (size_t)sub * S + 16 * u);
        // scalars, spread over the octet
        if (ol < P) {
            B.land[(size_t)g * P + ol] = gs.land[ol];
            B.army_total[(size_t)g * P + ol] = gs.tot[ol];
        }
        if (ol == (P & 7)) { B.turn[g] = gs.turn; B.alive[g] = (uint8_t)gs.alive; }
        if (ol == ((P + 1) & 7) && (flags & F_DIGEST) && B.obs_digest) B.obs_digest[g] = gs.digest;
        // the bitboard cache of the register-resident step kernel (generals_step.cuh): own[p], army >= 2,
        // structure, mountain; words past the board are 0 (all ones in the mountain row)
        if (B.bitboards) {
            uint32_t *bb = B.bitboards + (size_t)g * (size_t)(P + 3) * (size_t)BW;
            for (int u = ol; u < (P + 3) * BW; u += LPG) {
                const int row = u / BW, j = u - row * BW;
                const int m = row < P ? row : (row == P ? R_A2 : (row == P + 1 ? R_STR : R_MTN));
                bb[u] = j < NW ? mrow(m, sub)[j] : (row == P + 2 ? 0xFFFFFFFFu : 0u);
            }
        }
    }
}

}  // namespace gen
