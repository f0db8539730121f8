// generals_step.cuh -- the per-step kernel of gen_step (a2..a12 of SURVEY.md section 8, one turn per launch).
//
// REGISTER-RESIDENT design.  The three state planes are never staged in shared memory: what the rules
// need of them lives in the bitboard cache gen_buffers.bitboards ((P + 3) rows of one bit per cell per
// game: own[p], army >= 2, structure, mountain), which every kernel of the library keeps current.
//   * load: one TMA bulk copy per warp brings the cache rows of its 4 games (400 B each at 24x24 1v1)
//     into shared memory; the planes stay in HBM / L2;
//   * rules (sampler, moves, capture, growth, termination) run on the rows; the handful of army cells a
//     move or a structure's growth touches are read and written in global memory directly;
//   * emit: every lane reads its 8-cell chunks of the planes once, straight into registers (16 / 8-byte
//     coalesced loads), masks them with each player's fog row and streams the observation planes out.
// Shared memory per game drops from 3.3 KB to about 0.7 KB, so a whole 16,384-game batch is resident on
// the 148 SMs at once (one wave), and nothing is rebuilt from the planes per step.
//
// Same thread mapping as generals_kernels.cuh: a warp owns 4 consecutive games, an octet of 8 lanes one
// game; word passes split the octet by player; lane 0 of the octet runs the serial rules.  Same rules
// text (section IV, readings R1..R32 of DESIGN.md); parity with the oracle is bit-exact.
// Not served here (the host falls back to the staged kernel): observation digest, K > 1, gen_reset /
// gen_observe / gen_sample.
#pragma once
#include "generals_kernels.cuh"

namespace gen {

#ifdef GEN_TRACE  // development only: per-warp timeline (globaltimer at each mark), read by gen_debug_trace_<id>
constexpr int TRACE_MARKS = 16, TRACE_WARPS = 8192;
static __device__ unsigned long long g_trace[TRACE_WARPS * TRACE_MARKS];
__device__ __forceinline__ unsigned long long gtimer() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}
#define GEN_TRACE_MARK(k)                                                                         \
    do {                                                                                          \
        __syncwarp();                                                                             \
        if (lane == 0 && trace_w < TRACE_WARPS) g_trace[trace_w * TRACE_MARKS + (k) + 1] = gtimer(); \
    } while (0)
#else
#define GEN_TRACE_MARK(k)
#endif

struct StepGame {  // per-game scalars in shared memory
    int32_t turn, winner;
    uint32_t alive, done, episode, flags, sat;
    int32_t rew_bits;
    int32_t tot[8], land[8], act[8], gcell[8];
    uint32_t best[8], best_ok;  // BIAS: largest owned stack per player from gen_buffers.stack_cache, and whether it is current
    uint32_t rdirty[2];         // cache rows own[0..P-1], army >= 2: bit r * (BW / 8) + s = 32-byte sector s of row r changed
};

enum : uint32_t {
    SG_RESET = 1u << 0,      // auto-reset: regenerate the board in this call
    SG_FROZEN = 1u << 1,     // finished game without auto-reset (R31)
    SG_GROW_EVEN = 1u << 2,  // owned structures +1 this turn
    SG_GROW_TICK = 1u << 3,  // all owned cells +1 this turn
    SG_STATIC_DIRTY = 1u << 4,  // structure / mountain rows changed (regenerated): write them back too
    SG_ROWS_DIRTY = 1u << 5,    // own / army >= 2 rows changed wholesale (land transfer, 50-turn tick): write them all back
};

// ================================================================================================
// NP = bound of the player loops; CH x CW > 0: board size fixed at compile time and P == NP; MAXT / MINB:
// launch bounds (threads per CTA, resident CTAs per SM the register allocation must allow).
// BIAS: the build for the biased policy (R25): the observation pass also finds each player's largest owned stack and
// leaves it in gen_buffers.stack_cache for the next turn's sampler (which then does not scan the army plane).
template <int NP, int CH, int CW, int MAXT, int MINB, bool OFFICIAL, bool BIAS>
__global__ void __launch_bounds__(MAXT, MINB) k_step(const __grid_constant__ KParams kp) {
    constexpr bool FIXED = CH > 0;
    constexpr int LPP = LPG / NP;
    static_assert(!BIAS || NP < LPG, "lane P of the octet carries the stamp of gen_buffers.stack_cache");
    extern __shared__ __align__(128) unsigned char smem[];
    const int tid = threadIdx.x;
    const uint32_t lane = tid & 31u;
    const int wic = tid >> 5;
    const int ol = (int)(lane & (LPG - 1)), sub = (int)(lane / LPG);
    const uint32_t gmask = ((1u << LPG) - 1u) << (sub * LPG);
    const int pl = ol / LPP, sl = ol % LPP;
    constexpr int cHW = CH * CW, cS = (cHW + 15) / 16 * 16, cNW = (cHW + 31) / 32;
    const int H = FIXED ? CH : kp.H, W = FIXED ? CW : kp.W, P = FIXED ? NP : kp.P;
    const int HW = FIXED ? cHW : kp.HW, S = FIXED ? cS : kp.S, NW = FIXED ? cNW : kp.NW;
    const int NC8 = FIXED ? cS / 8 : kp.NC8;
    const int BW = FIXED ? (cNW + 7) / 8 * 8 : kp.BW;
    const int WS = (NW + LPP - 1) / LPP;
    const uint32_t flags = kp.flags;  // F_SAMPLER is the only mode bit this kernel looks at
    const gen_buffers &B = kp.b;
    const int wg0 = (blockIdx.x * kp.WPC + wic) * GW;
    const int nwg = min(GW, kp.N - wg0);
    const bool gvalid = sub < nwg;
    const int g = wg0 + sub;
    const uint32_t allp = (1u << P) - 1u;
    const bool teams = (FIXED && NP == 2) ? false : kp.team_size > 1;

    uint32_t *s_nc0 = reinterpret_cast<uint32_t *>(smem) + 1, *s_ncL = s_nc0 + 34, *s_inb = s_nc0 + 68;
    unsigned char *wb = smem + kp.off_warp0 + (size_t)wic * kp.warp_bytes;
    // rows of a game: [cache rows of the warp's games: own[0..P-1], army >= 2, structure, mountain] [vis[0..P-1]]
    uint32_t *s_rows = reinterpret_cast<uint32_t *>(wb);
    uint32_t *s_vis = s_rows + GW * (P + 3) * BW;
    StepGame *s_game = reinterpret_cast<StepGame *>(wb + kp.w_game);
    const uint32_t bar = smem_u32(wb + kp.w_bar);
    unsigned char *s_scratch = wb + kp.w_scratch;  // one game's planes while it is regenerated
    const int R_A2 = P, R_STR = P + 1, R_MTN = P + 2;
    auto row = [&](int m, int lg) -> uint32_t * { return s_rows + (lg * (P + 3) + m) * BW; };
    auto row8 = [&](int m, int lg) -> unsigned char * { return reinterpret_cast<unsigned char *>(row(m, lg)); };
    auto vrow = [&](int p, int lg) -> uint32_t * { return s_vis + (lg * P + p) * BW; };
    auto team_mask = [&](int p) -> uint32_t {
        const int t = p / kp.team_size;
        return (((1u << kp.team_size) - 1u) << (t * kp.team_size)) & allp;
    };
    auto row_of = [&](int cell) -> int {
        return FIXED ? (int)((uint32_t)cell / (uint32_t)(FIXED ? CW : 1)) : (int)(((uint32_t)cell * kp.recipW) >> 16);
    };
    auto bit_of = [&](const uint32_t *r, int c) -> bool { return (r[c >> 5] >> (c & 31)) & 1u; };
    auto set_bit = [&](uint32_t *r, int c, bool on) {
        const uint32_t bit = 1u << (c & 31);
        if (on) r[c >> 5] |= bit; else r[c >> 5] &= ~bit;
    };
    // The dynamic cache rows (own[p], army >= 2) go back to HBM by 32-byte sector, and only the sectors a turn
    // changed: a move flips a handful of bits.  mark_row: word j of row m of game gs changed.
    auto mark_row = [&](StepGame &gs, int m, int j) {
        const int sct = m * (BW >> 3) + (j >> 3);
        if (FIXED && (NP + 1) * (((cNW + 7) / 8 * 8) >> 3) <= 32) gs.rdirty[0] |= 1u << sct;   // one word holds them all
        else gs.rdirty[sct >> 5] |= 1u << (sct & 31);
    };
    auto set_bit_row = [&](StepGame &gs, int lg, int m, int c, bool on) {  // set_bit on row m, recording a change
        uint32_t *r = row(m, lg);
        const uint32_t bit = 1u << (c & 31), old = r[c >> 5], now = on ? (old | bit) : (old & ~bit);
        if (now != old) { r[c >> 5] = now; mark_row(gs, m, c >> 5); }
    };

    // ================================================================ prologue
#ifdef GEN_TRACE
    const int trace_w = blockIdx.x * kp.WPC + wic;
    if (lane == 0 && trace_w < TRACE_WARPS) g_trace[trace_w * TRACE_MARKS] = gtimer();
#endif
    for (int t = tid; t < 34; t += blockDim.x) {
        const int j = t - 1;
        const bool in = j >= 0 && j < 32;
        s_nc0[j] = in ? kp.notcol0[j & 31] : 0u;
        s_ncL[j] = in ? kp.notcolL[j & 31] : 0u;
        s_inb[j] = in ? kp.inb[j & 31] : 0u;
    }
    // Launch chaining (gen_buffers.step_epoch = start[NG] | done[NG], one pair per group of 4 games).  Every warp
    // takes a ticket for its group: the number of earlier launches that started on it.  The trigger below comes after
    // the tickets of this CTA have been taken (their values have arrived), and the CTAs of the next launch are placed
    // only after every CTA of this one has triggered, so tickets are handed out in launch order without any host
    // counter (graph replays and eager launches mix freely).
    uint32_t ticket = 0;
    const int NG = (kp.N + 3) >> 2;
    if (kp.count) {
        if (lane == 0 && nwg > 0) ticket = atomicAdd(B.step_epoch + (wg0 >> 2), 1u);
        ticket = __shfl_sync(FULL, ticket, 0);
        __syncthreads();
    }
    pdl_launch_dependents();  // the next launch may be placed as CTAs of this one retire ...
    // ... and nothing of the previous launch is read before it has completed: the whole grid, or -- chained launches
    // -- the warps of earlier launches that owned this warp's games: done == ticket.  A record that does not arrive
    // (a foreign writer of the buffer) ends in the grid-wide wait, which is always sufficient.
    if (kp.chain && nwg > 0) {
        const uint32_t *rec = B.step_epoch + NG + (wg0 >> 2);
        uint32_t seen = 0;
        int spins = 0;
        if (lane == 0) {
            for (;;) {
                asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(rec) : "memory");
                if (seen == ticket || ++spins > (1 << 16)) break;
                __nanosleep(100);
            }
            asm volatile("fence.proxy.async.global;" ::: "memory");  // the cache rows are read by the async proxy (TMA)
        }
        seen = __shfl_sync(FULL, seen, 0);
        if (seen != ticket) pdl_wait();
    } else {
        pdl_wait();
    }
    if (nwg > 0 && lane == 0) {
        mbar_init(bar, 1);
        const uint32_t bytes = (uint32_t)nwg * (uint32_t)(P + 3) * (uint32_t)BW * 4u;
        mbar_expect_tx(bar, bytes);
        bulk_g2s(smem_u32(s_rows), B.bitboards + (size_t)wg0 * (size_t)(P + 3) * (size_t)BW, bytes, bar);
    }
    if (gvalid) {  // per-game scalars: every lane issues all eight loads (one round trip), then the octet scatters
        StepGame &gs = s_game[sub];
        const size_t gp = (size_t)g * P + (size_t)min(ol, P - 1);
        const int32_t v_tot = __ldcg(B.army_total + gp), v_land = __ldcg(B.land + gp);
        const int32_t v_gc = __ldcg(B.general_cell + gp);
        const int32_t v_turn = __ldcg(B.turn + g);
        const uint32_t v_ep = __ldcg(B.episode + g), v_alive = __ldcg(B.alive + g), v_done = __ldcg(B.done + g);
        const int32_t v_win = __ldcg(B.winner + g);
        if (ol < P) { gs.tot[ol] = v_tot; gs.land[ol] = v_land; gs.gcell[ol] = v_gc; }
        if (ol == 0) { gs.turn = v_turn; gs.episode = v_ep; }
        if (ol == 1) { gs.alive = v_alive; gs.done = v_done; gs.winner = v_win; }
        if (ol == 2) { gs.flags = 0; gs.sat = 0; gs.rew_bits = 0; gs.rdirty[0] = 0; gs.rdirty[1] = 0; }
        if constexpr (BIAS) {
            const bool use = B.stack_cache && kp.stack_ok;  // the host vouches for the cache (generals_api.cu: launch)
            const uint32_t v_st = use ? __ldcg(B.stack_cache + (size_t)g * (P + 1) + min(ol, P)) : 0u;
            if (ol < P) gs.best[ol] = v_st;
            if (ol == P) gs.best_ok = (use && v_st == kp.global_step0) ? 1u : 0u;
        }
    }
    __syncthreads();  // the only CTA barrier: tables and the mbarrier init are visible
    if (nwg <= 0) return;
    GEN_TRACE_MARK(0);  // scalars + barrier
    mbar_wait(bar, 0);
    if (lane == 0) {
        // The planes of the warp's games are contiguous: start them on their way from HBM to L2 now (after the
        // small latency-critical loads above, so that those do not queue behind 9 KB of bulk traffic per warp);
        // the rules below run while they travel and the emit pass finds them in L2.
        const uint32_t cells = (uint32_t)nwg * (uint32_t)S;
        l2_prefetch(B.army + (size_t)wg0 * S, 2u * cells);
        l2_prefetch(B.owner + (size_t)wg0 * S, cells);
        l2_prefetch(B.terrain + (size_t)wg0 * S, cells);
    }
    GEN_TRACE_MARK(1);  // cache rows arrived

    // ---------------------------------------------------------------- a12: valid-action sampler (R24)
    // As in the staged kernel: the LPP lanes (pl, 0..LPP-1) of the octet serve player pl and split the NW
    // words; the valid list is ordered (direction, cell).  The four "target is free" masks are formed on
    // the fly from the mountain row (sliding window of three words).
    // No bounds test (it compiled to a divergent branch: 6 % of the kernel's instructions at 12 active threads): j runs
    // from -1 to NW, where s_inb[j] = 0 (guard words at both ends of the table; words past the board are 0 anyway) and
    // mtn[j] is some word of the warp's own shared memory.
    auto freew = [&](const uint32_t *mtn, int j) -> uint32_t { return ~mtn[j] & s_inb[j]; };
    auto sample = [&](int lg, uint32_t gstep) -> int {
        const int p = min(pl, P - 1);
        const uint32_t gid = kp.gid_base + (uint32_t)(wg0 + lg);
        uint32_t w[4];
        philox(0u, gid, gstep, (DOM_ACTION << 24) | (uint32_t)p, kp.key0, kp.key1, w);
        const uint32_t *own = row(p, lg), *a2 = row(R_A2, lg), *mtn = row(R_MTN, lg);
        const int js = sl * WS, je = min(js + WS, NW);
        uint32_t ln01 = 0, ln23 = 0;
        {
            uint32_t fp = freew(mtn, js - 1), fc = freew(mtn, js);
            for (int j = js; j < je; ++j) {
                const uint32_t fn = freew(mtn, j + 1);
                const uint32_t src = own[j] & a2[j];
                const uint32_t up = __funnelshift_lc(fp, fc, W), dn = __funnelshift_rc(fc, fn, W);
                const uint32_t lf = __funnelshift_l(fp, fc, 1) & s_nc0[j], rt = __funnelshift_r(fc, fn, 1) & s_ncL[j];
                ln01 += (uint32_t)__popc(src & up) | ((uint32_t)__popc(src & dn) << 16);
                ln23 += (uint32_t)__popc(src & lf) | ((uint32_t)__popc(src & rt) << 16);
                fp = fc; fc = fn;
            }
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
        if (kp.bias_thr) {  // uniform branch: the biased policy of config 4 (R25)
            // largest owned stack, ties -> lowest cell index: max of (army + 1) << 10 | (1023 - cell).  The army
            // plane stays in HBM / L2 in this kernel: every lane reads the 8-cell vectors of its words that hold an
            // owned cell (four independent 16-byte loads per word), compares in registers, the player's lanes reduce.
            const int16_t *Ag = B.army + (size_t)(wg0 + lg) * S;
            uint32_t best = 0;
            const bool cached = BIAS && s_game[lg].best_ok != 0;  // left by the previous turn's observation pass
            if (cached) best = s_game[lg].best[p];
            for (int j = cached ? je : js; j < je; ++j) {
                const uint32_t m = own[j] & s_inb[j];
                uint4 v[4];
#pragma unroll
                for (int q = 0; q < 4; ++q)
                    v[q] = ((m >> (8 * q)) & 0xFFu) ? __ldcg(reinterpret_cast<const uint4 *>(Ag + 32 * j + 8 * q))
                                                    : make_uint4(0u, 0u, 0u, 0u);
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const uint32_t mb = (m >> (8 * q)) & 0xFFu;
                    if (!mb) continue;
                    const uint32_t a[4] = {v[q].x, v[q].y, v[q].z, v[q].w};
#pragma unroll
                    for (int e = 0; e < 8; ++e) {
                        const uint32_t army = (a[e >> 1] >> (16 * (e & 1))) & 0xFFFFu;
                        const int c = 32 * j + 8 * q + e;
                        if ((mb >> e) & 1u) best = max(best, ((army + 1u) << 10) | (uint32_t)(1023 - c));
                    }
                }
            }
#pragma unroll
            for (int o = LPP / 2; o >= 1; o >>= 1) best = max(best, __shfl_xor_sync(gmask, best, o));
            if (!decided && w[3] < kp.bias_thr && best) {
                const int bc = 1023 - (int)(best & 1023u), jb = bc >> 5, bb = bc & 31;
                const uint32_t fp = freew(mtn, jb - 1), fc = freew(mtn, jb), fn = freew(mtn, jb + 1);
                const uint32_t src = (own[jb] & a2[jb]) >> bb;
                const uint32_t okw[4] = {__funnelshift_lc(fp, fc, W), __funnelshift_rc(fc, fn, W),
                                         __funnelshift_l(fp, fc, 1) & s_nc0[jb], __funnelshift_r(fc, fn, 1) & s_ncL[jb]};
                uint32_t vb = 0;
#pragma unroll
                for (int dd = 0; dd < 4; ++dd) vb |= ((src & (okw[dd] >> bb)) & 1u) << dd;
                if (vb) {
                    const int dd = nth_bit(vb, mulhi32(w[1], (uint32_t)__popc(vb)));
                    action = bc * 9 + 1 + 2 * dd + half;
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
                const uint32_t fp = freew(mtn, j - 1), fc = freew(mtn, j), fn = freew(mtn, j + 1);
                const uint32_t okd = d == 0 ? __funnelshift_lc(fp, fc, W)
                                   : d == 1 ? __funnelshift_rc(fc, fn, W)
                                   : d == 2 ? (__funnelshift_l(fp, fc, 1) & s_nc0[j])
                                            : (__funnelshift_r(fc, fn, 1) & s_ncL[j]);
                vw = own[j] & a2[j] & okd;
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
    // The rows answer every question but the two army values, which are read from and written to the
    // army plane in global memory (ld.global.cg: L2 only, so that the emit pass of the other lanes sees them).
    auto owner_of = [&](int lg, int c) -> int {
        int t = -1;
#pragma unroll
        for (int q = 0; q < NP; ++q)
            if (q < P && bit_of(row(q, lg), c)) t = q;
        return t;
    };
    // Movers i0 .. i1 - 1 of the turn's order; the call that reaches the last mover also advances the turn counter.
    auto play_moves = [&](int lg, int i0, int i1) {
        StepGame &gs = s_game[lg];
        const int gg = wg0 + lg;
        int16_t *A = B.army + (size_t)gg * S;
        int8_t *O = B.owner + (size_t)gg * S, *Tr = B.terrain + (size_t)gg * S;
        uint32_t *a2row = row(R_A2, lg);
        const uint32_t *mtn = row(R_MTN, lg);
        const int first = (kp.rule_flags & GEN_RULE_ROTATE_PRIORITY) ? (gs.turn % P) : 0;
        int bad = 0;  // non-pass actions that are not applied (diagnostic counter invalid_actions)
        for (int i = i0; i < i1; ++i) {
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
            // R5, R10: own the source, army >= 2 (the row is exact), target no mountain
            if (!bit_of(row(p, lg), cell) || !bit_of(a2row, cell) || bit_of(mtn, dst)) { ++bad; continue; }
            const int asrc = __ldcg(A + cell), d = __ldcg(A + dst);
            const int m = half ? (asrc >> 1) : (asrc - 1);  // R4
            const int nsrc = asrc - m;
            const int t = owner_of(lg, dst);
            const bool dst_general = t >= 0 && gs.gcell[t] == dst;
            int ndst, nown = t;
            bool captured = false;
            const bool ally = teams && t >= 0 && t != p && ((team_mask(p) >> t) & 1u);
            if (t == p || ally) {  // R8 / P:L97, R19
                ndst = d + m;
                int lost = 0;
                if (ndst > 32767) { lost = ndst - 32767; ndst = 32767; gs.sat += 1; }  // R21
                int holder = p;
                if (ally) {
                    if (!dst_general) { nown = p; gs.tot[p] += d; gs.tot[t] -= d; }
                    else { gs.tot[p] -= m; gs.tot[t] += m; holder = t; }
                }
                if (lost) gs.tot[holder] -= lost;
            } else if (m > d) {
                ndst = m - d;
                nown = p;
                captured = dst_general;  // R11, R12
                gs.tot[p] -= d;
                if (t >= 0) gs.tot[t] -= d;
            } else {
                ndst = d - m;  // tie -> 0, previous owner keeps the cell
                gs.tot[p] -= m;
                if (t >= 0) gs.tot[t] -= m;
            }
            A[cell] = (int16_t)nsrc;
            A[dst] = (int16_t)ndst;
            set_bit_row(gs, lg, R_A2, cell, nsrc >= 2);
            set_bit_row(gs, lg, R_A2, dst, ndst >= 2);
            if (nown != t) {
                O[dst] = (int8_t)nown;
                set_bit_row(gs, lg, nown, dst, true);
                gs.land[nown] += 1;
                if (t >= 0) { set_bit_row(gs, lg, t, dst, false); gs.land[t] -= 1; }
            }
            if (captured) {  // a4: land transfer (R11); the general becomes a city
                const int q = t;
                gs.flags |= SG_ROWS_DIRTY;
                Tr[dst] = (int8_t)T_CITY;
                gs.alive &= ~(1u << q);
                gs.gcell[q] = -1;
                B.general_cell[(size_t)gg * P + q] = -1;
                const bool fl = (kp.rule_flags & GEN_RULE_CAPTURE_HALF_FLOOR) != 0;
                uint32_t *oq = row(q, lg), *op = row(p, lg);
                int moved = 0;
                for (int j = 0; j < NW; ++j) {
                    uint32_t wq = oq[j];
                    if (wq == 0) continue;
                    op[j] |= wq;
                    oq[j] = 0;
                    uint32_t a2w = a2row[j];
                    while (wq) {
                        const int b = __ffs(wq) - 1;
                        wq &= wq - 1;
                        const int c = 32 * j + b;
                        O[c] = (int8_t)p;
                        const int av = __ldcg(A + c);
                        const int nv = fl ? (av >> 1) : ((av + 1) >> 1);
                        A[c] = (int16_t)nv;
                        moved += nv;
                        a2w = nv >= 2 ? (a2w | (1u << b)) : (a2w & ~(1u << b));
                    }
                    a2row[j] = a2w;
                }
                gs.tot[p] += moved;
                gs.tot[q] = 0;
                gs.land[p] += gs.land[q];
                gs.land[q] = 0;
            }
        }
        if (bad && B.invalid_actions) B.invalid_actions[gg] += (uint32_t)bad;
        if (i1 < P) return;
        // a6: turn counter; growth itself is applied by the next parallel pass (R1, R2, R3)
        const int turn = gs.turn + 1;
        gs.turn = turn;
        uint32_t gflags = 0;
        if ((turn & 1) == 0) gflags |= SG_GROW_EVEN;
        if (turn % 50 == 0) gflags |= SG_GROW_TICK;
        if (gflags) gs.flags |= gflags;
    };

    // ---------------------------------------------------------------- a6: growth (octet), army plane in global
    // tick turns (every 50th, always even): +1 on owned cells, +1 more on owned structures (R2)
    auto grow_tick = [&](int lg) {
        StepGame &gs = s_game[lg];
        int16_t *A = B.army + (size_t)(wg0 + lg) * S;
        for (int ch = ol; ch < NC8; ch += LPG) {
            const uint32_t sb = row8(R_STR, lg)[ch];
            uint32_t ob[NP], ownedb = 0;
#pragma unroll
            for (int p = 0; p < NP; ++p) { ob[p] = p < P ? row8(p, lg)[ch] : 0u; ownedb |= ob[p]; }
            const uint32_t e = sb & ownedb;
            const uint32_t t = (kp.rule_flags & GEN_RULE_TICK_PLAIN_ONLY) ? (ownedb & ~sb) : ownedb;
            if ((e | t) == 0) continue;
            uint4 *ap = reinterpret_cast<uint4 *>(A + 8 * ch);
            uint4 a = __ldcg(ap);
            uint32_t aw[4] = {a.x, a.y, a.z, a.w};
            bool sat = false;
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const uint32_t lo = ((e >> (2 * k)) & 1u) + ((t >> (2 * k)) & 1u);
                const uint32_t hi = ((e >> (2 * k + 1)) & 1u) + ((t >> (2 * k + 1)) & 1u);
                aw[k] += lo | (hi << 16);
                sat |= (aw[k] & 0x80008000u) != 0;
            }
            int lost[NP];
#pragma unroll
            for (int p = 0; p < NP; ++p) lost[p] = 0;
            if (sat) {  // R21: every +1 that would pass 32767 is one saturation event, charged to the owner
                int ev = 0;
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    uint32_t v = (i & 1) ? (aw[i >> 1] >> 16) : (aw[i >> 1] & 0xFFFFu);
                    if (v > 32767u) {
                        const int over = (int)(v - 32767u);
                        ev += over;
#pragma unroll
                        for (int p = 0; p < NP; ++p)
                            if ((ob[p] >> i) & 1u) lost[p] += over;
                        aw[i >> 1] = (i & 1) ? ((aw[i >> 1] & 0xFFFFu) | (32767u << 16))
                                             : ((aw[i >> 1] & 0xFFFF0000u) | 32767u);
                    }
                }
                atomicAdd(&gs.sat, (uint32_t)ev);
            }
            a.x = aw[0]; a.y = aw[1]; a.z = aw[2]; a.w = aw[3];
            *ap = a;
            row8(R_A2, lg)[ch] = (unsigned char)ge2_bits(a);
#pragma unroll
            for (int p = 0; p < NP; ++p) {
                const int inc = __popc(e & ob[p]) + __popc(t & ob[p]) - lost[p];
                if (p < P && inc) atomicAdd(&gs.tot[p], inc);
            }
        }
    };
    // even turns that are no tick: +1 on the few owned structures, found by bit iteration
    auto grow_structures = [&](int lg) {
        StepGame &gs = s_game[lg];
        int16_t *A = B.army + (size_t)(wg0 + lg) * S;
        for (int j = ol; j < NW; j += LPG) {
            const uint32_t sw = row(R_STR, lg)[j];
            if (sw == 0) continue;
            uint32_t a2w = row(R_A2, lg)[j];
            bool changed = false;
            for (int p = 0; p < P; ++p) {
                uint32_t m = sw & row(p, lg)[j];
                if (m == 0) continue;
                int inc = 0;
                // Fast path, no load: a cell of a player whose whole army is below 32767 cannot saturate, and a cell
                // with army >= 2 keeps its bit: +1 as a fire-and-forget reduction on the 32-bit word that holds it.
                if (gs.tot[p] <= 32766) {
                    uint32_t f = m & a2w;
                    m &= ~a2w;
                    inc = __popc(f);
                    while (f) {
                        const int b = __ffs(f) - 1;
                        f &= f - 1;
                        const int c = 32 * j + b;
                        atomicAdd(reinterpret_cast<unsigned int *>(A + (c & ~1)), (c & 1) ? 0x10000u : 1u);
                    }
                }
                while (m) {
                    const int b = __ffs(m) - 1;
                    m &= m - 1;
                    const int c = 32 * j + b, av = __ldcg(A + c);
                    if (av >= 32767) { atomicAdd(&gs.sat, 1u); continue; }  // R21
                    A[c] = (int16_t)(av + 1);
                    inc += 1;
                    if (av == 1) { a2w |= 1u << b; changed = true; }
                }
                if (inc) atomicAdd(&gs.tot[p], inc);
            }
            if (changed) {
                row(R_A2, lg)[j] = a2w;
                const int sct = R_A2 * (BW >> 3) + (j >> 3);
                atomicOr(&gs.rdirty[sct >> 5], 1u << (sct & 31));
            }
        }
    };

    // ---------------------------------------------------------------- a7-a9: end of turn, one lane per game
    auto write_result = [&](int gg, int rew_bits, uint32_t done, int winner) {
        int8_t *rw = B.reward + (size_t)gg * P;
        if (rew_bits == 0x5555 >> (16 - 2 * P) && (P == 2 || P == 4 || P == 8)) {  // all zero: one store
            if (P == 2) *reinterpret_cast<uint16_t *>(rw) = 0;
            else if (P == 4) *reinterpret_cast<uint32_t *>(rw) = 0;
            else *reinterpret_cast<uint2 *>(rw) = make_uint2(0u, 0u);
        } else {
            for (int p = 0; p < P; ++p) rw[p] = (int8_t)(((rew_bits >> (2 * p)) & 3) - 1);
        }
        B.done[gg] = (uint8_t)done;
        B.winner[gg] = (int8_t)winner;
        // gen_step_host[_async] with pinned result arrays: the same values straight to the host (posted writes through
        // the mapped aliases; the four games of a warp are adjacent, so a warp sends 4 * P + 4 contiguous bytes) --
        // no second kernel behind the step
        if (kp.mirror_reward) {
            int8_t *hr = kp.mirror_reward + (size_t)gg * P;
            if (P == 2) *reinterpret_cast<uint16_t *>(hr) = (uint16_t)(((uint32_t)(uint8_t)(((rew_bits >> 0) & 3) - 1)) |
                                                                        ((uint32_t)(uint8_t)(((rew_bits >> 2) & 3) - 1) << 8));
            else for (int p = 0; p < P; ++p) hr[p] = (int8_t)(((rew_bits >> (2 * p)) & 3) - 1);
        }
        if (kp.mirror_done) kp.mirror_done[gg] = (uint8_t)done;
    };
    auto finish_turn = [&](int lg) {
        StepGame &gs = s_game[lg];
        const int gg = wg0 + lg;
        if (gs.sat) { B.sat_events[gg] += gs.sat; gs.sat = 0; }
        const int zero_bits = 0x5555 >> (16 - 2 * P);
        const bool truncated_now = kp.max_turns > 0 && gs.turn >= kp.max_turns;
        if (gs.alive == allp && !truncated_now && kp.n_teams > 1) {  // the common case: nothing ends
            gs.done = 0;
            gs.winner = -1;
            write_result(gg, zero_bits, 0u, -1);
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
        write_result(gg, rew_bits, gs.done, gs.winner);
        if (gs.done) {
            B.episodes_done[gg] += 1;
            if (truncated) B.truncations[gg] += 1;
            if (kp.auto_reset) {  // a9 (R17)
                gs.episode += 1;
                B.episode[gg] = gs.episode;
                gs.flags |= SG_RESET;
            }
        }
    };

    // ---------------------------------------------------------------- a9 + a1: regenerate game lg (whole warp)
    // The generator fills one game's planes in the warp's scratch; the rows are gathered from them and the
    // planes copied out to HBM.
    auto regenerate = [&](int lg) {
        StepGame &gs = s_game[lg];
        const int gg = wg0 + lg;
        int16_t *sA = reinterpret_cast<int16_t *>(s_scratch);
        int8_t *sO = reinterpret_cast<int8_t *>(s_scratch + 2 * S), *sT = reinterpret_cast<int8_t *>(s_scratch + 3 * S);
        generate_board<NP, OFFICIAL>(kp, lane, kp.gid_base + (uint32_t)gg, gs.episode, sA, sO, sT,
                                     B.general_cell + (size_t)gg * P,
                                     B.play_size ? B.play_size + 2 * (size_t)gg : nullptr);
        const int rb = 4 * BW;  // row stride in bytes
        unsigned char *rows = row8(0, lg);
        for (int ch = (int)lane; ch < rb; ch += 32) {
            if (ch < NC8) {
                const uint2 o = *reinterpret_cast<const uint2 *>(sO + 8 * ch);
                const uint2 t = *reinterpret_cast<const uint2 *>(sT + 8 * ch);
                const uint4 a = *reinterpret_cast<const uint4 *>(sA + 8 * ch);
#pragma unroll
                for (int p = 0; p < NP; ++p)
                    if (p < P) {
                        const uint32_t pat = 0x01010101u * (uint32_t)p;
                        rows[p * rb + ch] = (unsigned char)gather8<0>(eq_bytes(o.x, pat), eq_bytes(o.y, pat));
                    }
                const uint32_t hx = t.x >> 1, hy = t.y >> 1;  // terrain: mountain = 01, structure = 1x
                rows[R_MTN * rb + ch] = (unsigned char)gather8<0>(t.x & ~hx, t.y & ~hy);
                rows[R_STR * rb + ch] = (unsigned char)gather8<0>(hx, hy);
                rows[R_A2 * rb + ch] = (unsigned char)ge2_bits(a);
            } else {
                for (int p = 0; p < P; ++p) rows[p * rb + ch] = 0;
                rows[R_MTN * rb + ch] = 0xFF;
                rows[R_STR * rb + ch] = 0;
                rows[R_A2 * rb + ch] = 0;
            }
        }
        const size_t gbase = (size_t)gg * S;
        for (int u = (int)lane; u < S / 8; u += 32)
            *reinterpret_cast<uint4 *>(B.army + gbase + 8 * u) = *reinterpret_cast<const uint4 *>(sA + 8 * u);
        for (int u = (int)lane; u < S / 16; u += 32) {
            *reinterpret_cast<uint4 *>(B.owner + gbase + 16 * u) = *reinterpret_cast<const uint4 *>(sO + 16 * u);
            *reinterpret_cast<uint4 *>(B.terrain + gbase + 16 * u) = *reinterpret_cast<const uint4 *>(sT + 16 * u);
        }
        if (lane == 0) {
            gs.turn = 0;
            gs.alive = allp;
            gs.flags = (gs.flags & ~SG_RESET) | SG_STATIC_DIRTY;
            for (int p = 0; p < P; ++p) {
                gs.tot[p] = 1;
                gs.land[p] = 1;
                gs.gcell[p] = B.general_cell[(size_t)gg * P + p];
            }
        }
        __syncwarp();
    };

    // ---------------------------------------------------------------- a10: fog of war (all players at once)
    auto compute_vis = [&](int lg) {
        if (pl >= P) return;
        const int js = sl * WS, je = min(js + WS, NW);
        if (js >= je) return;
        uint32_t *vr = vrow(pl, lg);
        const uint32_t *own = row(pl, lg);
        const uint32_t members = teams ? team_mask(pl) : 0u;
        auto tw = [&](int j) -> uint32_t {
            if ((unsigned)j >= (unsigned)NW) return 0u;
            if (!teams) return own[j];
            uint32_t tm = 0;
            for (int q = 0; q < P; ++q)
                if ((members >> q) & 1u) tm |= row(q, lg)[j];
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
    // Lane ol owns the 8-cell chunks ol, ol + 8, ...: per chunk the octet covers full 128 / 64-byte lines.
    // Two passes, each with ALL its global loads issued before the first use (memory-level parallelism: one
    // round trip per pass instead of one per chunk): (A) the army plane, 16 bytes per chunk; (B) owner and
    // terrain, 8 + 8 bytes.  Every chunk is masked once per player with that player's fog byte and leaves
    // as one 16-byte and three 8-byte streaming stores.
    auto emit_planes = [&](int lg) {
#ifndef GEN_EB
#define GEN_EB 9
#endif
        constexpr int EB = FIXED ? ((cS / 8 + LPG - 1) / LPG < GEN_EB ? (cS / 8 + LPG - 1) / LPG : GEN_EB) : 4;  // chunks per batch
        const size_t gbase = (size_t)(wg0 + lg) * (size_t)S;
        const size_t obase = gbase * (size_t)P;
        const unsigned char *__restrict__ ga = reinterpret_cast<const unsigned char *>(B.army + gbase) + 16 * ol;
        const unsigned char *__restrict__ go = reinterpret_cast<const unsigned char *>(B.owner + gbase) + 8 * ol;
        const unsigned char *__restrict__ gt = reinterpret_cast<const unsigned char *>(B.terrain + gbase) + 8 * ol;
        unsigned char *__restrict__ oa = reinterpret_cast<unsigned char *>(B.obs_army + obase) + 16 * ol;
        unsigned char *__restrict__ oo = reinterpret_cast<unsigned char *>(B.obs_owner + obase) + 8 * ol;
        unsigned char *__restrict__ ot = reinterpret_cast<unsigned char *>(B.obs_terrain + obase) + 8 * ol;
        unsigned char *__restrict__ ov = reinterpret_cast<unsigned char *>(B.obs_vis + obase) + 8 * ol;
        unsigned char *__restrict__ op = reinterpret_cast<unsigned char *>(B.obs_packed + obase) + 8 * ol;
        const bool packed = B.obs_packed != nullptr;
        const unsigned char *sv = reinterpret_cast<const unsigned char *>(vrow(0, lg)) + ol;
        const int nit = (NC8 - ol + LPG - 1) / LPG;
        uint32_t bb[NP];  // BIAS: largest owned stack per player among this lane's chunks
#pragma unroll
        for (int p = 0; p < NP; ++p) bb[p] = 0;
        for (int i0 = 0; i0 < nit; i0 += EB) {
            // ---- pass A: army
            uint4 a[EB];
#pragma unroll
            for (int k = 0; k < EB; ++k)
                if (i0 + k < nit) a[k] = __ldcg(reinterpret_cast<const uint4 *>(ga + 128 * (i0 + k)));
#pragma unroll
            for (int k = 0; k < EB; ++k) {
                if (i0 + k >= nit) break;
                const int i = i0 + k;
#pragma unroll
                for (int p = 0; p < NP; ++p) {
                    if (p >= P) break;
                    const uint32_t vb = sv[4 * BW * p + 8 * i];
                    const uint32_t s0 = nib_sign(vb & 15u), s1 = nib_sign(vb >> 4);
                    uint4 xa;
                    xa.x = a[k].x & prmt(s0, 0u, 0x9988u); xa.y = a[k].y & prmt(s0, 0u, 0xBBAAu);
                    xa.z = a[k].z & prmt(s1, 0u, 0x9988u); xa.w = a[k].w & prmt(s1, 0u, 0xBBAAu);
                    __stcs(reinterpret_cast<uint4 *>(oa + 2 * (size_t)p * (size_t)S + 128 * i), xa);
                    if constexpr (BIAS) {  // (army + 1) << 10 | (1023 - cell): max = largest stack, ties to the lowest cell
                        const uint32_t ob = row8(p, lg)[ol + LPG * i];
                        if (ob) {
                            const uint32_t aa[4] = {a[k].x, a[k].y, a[k].z, a[k].w};
#pragma unroll
                            for (int e = 0; e < 8; ++e) {
                                const uint32_t army = (aa[e >> 1] >> (16 * (e & 1))) & 0xFFFFu;
                                const uint32_t key = ((army + 1u) << 10) | (uint32_t)(1023 - (8 * (ol + LPG * i) + e));
                                if ((ob >> e) & 1u) bb[p] = max(bb[p], key);
                            }
                        }
                    }
                }
            }
            // ---- pass B: owner, terrain, visibility -- three byte planes, or one packed byte (R33)
            uint2 o[EB], t[EB];
#pragma unroll
            for (int k = 0; k < EB; ++k)
                if (i0 + k < nit) {
                    o[k] = __ldcg(reinterpret_cast<const uint2 *>(go + 64 * (i0 + k)));
                    t[k] = __ldcg(reinterpret_cast<const uint2 *>(gt + 64 * (i0 + k)));
                }
            if (packed) {
#pragma unroll
                for (int k = 0; k < EB; ++k) {
                    if (i0 + k >= nit) break;
                    const int i = i0 + k;
                    // per byte: 0x80 | terrain << 4 | (owner + 2); owner + 2 on the low nibble cannot carry
                    const uint32_t qx = 0x80808080u | ((t[k].x << 4) & 0x30303030u) |
                                        (((o[k].x & 0x0F0F0F0Fu) + 0x02020202u) & 0x0F0F0F0Fu);
                    const uint32_t qy = 0x80808080u | ((t[k].y << 4) & 0x30303030u) |
                                        (((o[k].y & 0x0F0F0F0Fu) + 0x02020202u) & 0x0F0F0F0Fu);
#pragma unroll
                    for (int p = 0; p < NP; ++p) {
                        if (p >= P) break;
                        const uint32_t vb = sv[4 * BW * p + 8 * i];
                        const uint32_t m0 = prmt(nib_sign(vb & 15u), 0u, 0xBA98u), m1 = prmt(nib_sign(vb >> 4), 0u, 0xBA98u);
                        __stcs(reinterpret_cast<uint2 *>(op + (size_t)p * (size_t)S + 64 * i), make_uint2(qx & m0, qy & m1));
                    }
                }
                continue;
            }
#pragma unroll
            for (int k = 0; k < EB; ++k) {
                if (i0 + k >= nit) break;
                const int i = i0 + k;
#pragma unroll
                for (int p = 0; p < NP; ++p) {
                    if (p >= P) break;
                    const uint32_t vb = sv[4 * BW * p + 8 * i];
                    const uint32_t m0 = prmt(nib_sign(vb & 15u), 0u, 0xBA98u), m1 = prmt(nib_sign(vb >> 4), 0u, 0xBA98u);
                    uint2 xo, xt, xv;
                    xo.x = (o[k].x & m0) | (~m0 & 0xFEFEFEFEu); xo.y = (o[k].y & m1) | (~m1 & 0xFEFEFEFEu);
                    xt.x = (t[k].x & m0) | (~m0 & 0x04040404u); xt.y = (t[k].y & m1) | (~m1 & 0x04040404u);
                    xv.x = m0 & 0x01010101u; xv.y = m1 & 0x01010101u;
                    const size_t po = (size_t)p * (size_t)S;
                    __stcs(reinterpret_cast<uint2 *>(oo + po + 64 * i), xo);
                    __stcs(reinterpret_cast<uint2 *>(ot + po + 64 * i), xt);
                    __stcs(reinterpret_cast<uint2 *>(ov + po + 64 * i), xv);
                }
            }
        }
        if constexpr (BIAS) {
            if (B.stack_cache) {
                uint32_t mine = kp.global_step0 + 1u;  // lane P: the step at which this state will be sampled
#pragma unroll
                for (int p = 0; p < NP; ++p) {
#pragma unroll
                    for (int o = LPG / 2; o >= 1; o >>= 1) bb[p] = max(bb[p], __shfl_xor_sync(gmask, bb[p], o));
                    if (ol == p) mine = bb[p];
                }
                if (ol <= P) B.stack_cache[(size_t)(wg0 + lg) * (P + 1) + ol] = mine;
            }
        }
    };

    // ================================================================ the turn
    const uint32_t gstep = kp.global_step0;
    bool frozen = false;
    if (gvalid) {
        StepGame &gs = s_game[sub];
        frozen = !kp.auto_reset && gs.done != 0;  // R31
        int a = 0;
        if (!frozen) {
            if (flags & F_SAMPLER) a = sample(sub, gstep);
            else if (sl == 0 && pl < P) a = kp.actions[(size_t)g * P + pl];
        }
        if (sl == 0 && pl < P) {
            gs.act[pl] = a;
            if (B.actions_out) B.actions_out[(size_t)g * P + pl] = a;
        }
    }
    __syncwarp();
    GEN_TRACE_MARK(2);  // sampler
    if constexpr (NP > 2) {
        // One mover per divergent region.  The moves run on one lane per game while the other 28 lanes wait at the
        // region's convergence barrier; when that wait is long -- eight movers, two dependent L2 round trips each --
        // the waiting lanes were observed (ncu, k_step<8,32,32>: 16 active threads per instruction from here to the end
        // of the kernel, every store instruction issued twice and its sectors written in two parts) to be let go and
        // never to rejoin the moving lanes: __syncwarp() makes them wait for each other but does not merge them.
        // Short regions reconverge.
        for (int i = 0; i < P; ++i) {
            if (gvalid && ol == 0 && !frozen) play_moves(sub, i, i + 1);
            __syncwarp();
        }
        if (gvalid && ol == 0 && frozen) s_game[sub].flags |= SG_FROZEN;
    } else if (gvalid && ol == 0) {
        if (frozen) s_game[sub].flags |= SG_FROZEN;
        else play_moves(sub, 0, P);
    }
    __syncwarp();
    GEN_TRACE_MARK(3);  // moves
    if (gvalid) {
        const uint32_t gf = s_game[sub].flags;
        if (gf & SG_GROW_TICK) grow_tick(sub);
        else if (gf & SG_GROW_EVEN) grow_structures(sub);
    }
    __syncwarp();
    GEN_TRACE_MARK(4);  // growth
    bool want_reset = false;
    if (gvalid && ol == 0) {
        StepGame &gs = s_game[sub];
        if (frozen) write_result(g, 0x5555 >> (16 - 2 * P), gs.done, gs.winner);
        else finish_turn(sub);
        want_reset = (gs.flags & SG_RESET) != 0;
    }
    const uint32_t rs = __ballot_sync(FULL, want_reset);  // bit sub * LPG: game sub must be regenerated
    if (rs) {
        for (int lg = 0; lg < nwg; ++lg)
            if ((rs >> (lg * LPG)) & 1u) regenerate(lg);
    }
    __syncwarp();
    GEN_TRACE_MARK(5);  // end of turn (+ regeneration)
    // ---- store the cache rows and scalars now: they are final, and after the emit pass the warp can retire at once
    if (gvalid) {
        const StepGame &gs = s_game[sub];
        const int nrows = (gs.flags & SG_STATIC_DIRTY) ? P + 3 : P + 1;  // own[p] + army >= 2 (+ structure, mountain)
        const uint4 *src = reinterpret_cast<const uint4 *>(row(0, sub));
        uint4 *dst = reinterpret_cast<uint4 *>(B.bitboards + (size_t)g * (size_t)(P + 3) * (size_t)BW);
        if (!frozen) {
            const bool all = (gs.flags & (SG_STATIC_DIRTY | SG_ROWS_DIRTY | SG_GROW_TICK)) != 0;  // the tick rewrites army >= 2
            for (int u = ol; u < nrows * BW / 4; u += LPG)   // 16-byte unit u lies in sector u >> 1 (rows are BW / 8 sectors)
                if (all || ((gs.rdirty[u >> 6] >> ((u >> 1) & 31)) & 1u)) dst[u] = src[u];
        }
        if (ol < P) {
            B.land[(size_t)g * P + ol] = gs.land[ol];
            B.army_total[(size_t)g * P + ol] = gs.tot[ol];
            if (B.score_hist && !frozen)  // R34: slot (turn mod 512) of the scoreboard history ring
                *reinterpret_cast<int2 *>(B.score_hist + (((size_t)g * 512 + (size_t)(gs.turn & 511)) * P + ol) * 2) =
                    make_int2(gs.land[ol], gs.tot[ol]);
        }
        if (ol == (P & 7)) { B.turn[g] = gs.turn; B.alive[g] = (uint8_t)gs.alive; }
    }
    // ---- a10 + a11 (R32: the state at the end of the call)
    if (gvalid) compute_vis(sub);
    __syncwarp();
    GEN_TRACE_MARK(6);  // fog
    if (gvalid) emit_planes(sub);
    GEN_TRACE_MARK(7);  // emit
    if (kp.count) {  // everything this warp wrote for its games is ordered before the record the next launch waits for
        __syncwarp();
        if (lane == 0) {  // release at gpu scope: cumulative over the lanes' stores ordered by the __syncwarp above
            asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(B.step_epoch + NG + (wg0 >> 2)), "r"(ticket + 1u) : "memory");
            // A chained grid did not wait for its predecessor on the way in, so one of its warps does on the way
            // out: this grid cannot complete before the previous one has, and whatever follows in the stream (a
            // kernel that is not ours, a staged-kernel call) sees completed grids in stream order by construction.
            if (kp.chain && blockIdx.x == 0 && wic == 0) pdl_wait();
        }
    }

    GEN_TRACE_MARK(8);  // store
}

}  // namespace gen
