/*
 * generals_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, single-threaded CPU implementation of the batched Generals.io
 * environment step of arXiv 2606.23348 (section IV, "P:Lnn" = line nn
 * of /root/reference/PAPER.md).  It exists only so that tests/, bench.py's
 * cpu_baseline / --impl reference leg and __graft_entry__.smoke() can check the
 * CUDA path against something written straight from the paper.  It shares no
 * code, header, table or constant generator with paper_2606_23348_b200/csrc/;
 * neither side includes or imports the other.  The product path never calls it.
 *
 * Every rule is a straight loop over cells / players in the paper's order.
 * Readings of the paper where it is silent or ambiguous are the "R<n>" items
 * of DESIGN.md (section "Readings"); each use below names its R-number.
 *
 * Parity pins (tests/test_oracle_*.py, run with -m "not gpu"):
 *   philox4x32_10   : Random123 known-answer vectors (tests/golden/philox_kat.txt)
 *   splitmix64 keys : published first outputs of splitmix64(seed 0)
 *   step rules      : hand-worked examples W1..W11, closed forms C1..C3,
 *                     invariants I1..I7, brute force B1/B2, metamorphic M1/M2
 *   generator       : statistical + constraint checks, brute-force candidate lists
 *   official maps   : (R36) constraints of P:L79 re-checked with an independent shortest-path routine, Manhattan
 *                     closed form, tiny boards by hand (tests/test_oracle_mapgen.py)
 *   feature tensor  : (R35) hand-worked example W12 (tests/golden/features_worked_example.txt), channel identities,
 *                     closed form, an independent memory log (test_oracle_features.py); bfloat16 (R37): torch's conversion
 *   history windows : (R39) closed form C1 through a ring wrap with 1, 2 (free-for-all) and 2 (2v2) enemies,
 *                     and an independent per-turn log on sampled play with auto-reset (test_oracle_properties.py)
 *   sampler         : brute force "valid set == set of board-changing actions"
 * Parity unpinned BY THE PAPER (fixed by decree in DESIGN.md, the paper prints no
 * value that decides them): R6 move order, R11 rounding of the transferred half,
 * R16/R17 truncation + auto-reset convention, R18 fog encodings, R19 ally-general
 * exception, R20 n-player reward, R21 saturation, R24/R25/R30 stream layout.
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

enum { T_PLAIN = 0, T_MOUNTAIN = 1, T_CITY = 2, T_GENERAL = 3, T_FOG = 4 };
enum { OWNER_NEUTRAL = -1, OWNER_FOG = -2 };
enum { ARMY_MAX = 32767 };
enum { RULE_TICK_PLAIN_ONLY = 1, RULE_CAPTURE_HALF_FLOOR = 2, RULE_ROTATE_PRIORITY = 4 };
enum { DOM_SPAWN = 1, DOM_MOUNTAIN = 2, DOM_CITY = 3, DOM_ACTION = 4 };
enum { DONE_TERMINATED = 1, DONE_TRUNCATED = 2 };
enum { ORC_OBS_DIGEST = 0, ORC_OBS_EVERY_STEP = 1, ORC_OBS_NONE = 2 };

typedef struct {
    int32_t n_games, height, width, n_players, team_size;
    int32_t n_cities, city_army_lo, city_army_hi;
    int32_t spawn_dmin, spawn_dmax, spawn_exact;
    int32_t max_turns, auto_reset;
    uint32_t rule_flags, game_id_base, mountain_thr;
    uint32_t pass_thr, half_thr, bias_thr, pad_;
    uint64_t seed;
    int32_t map_mode;         /* 0 = synthetic generator (R30), 1 = official generator (R36) */
    int32_t n_cities_max;     /* R36: castle count uniform in [n_cities, n_cities_max]; 0 = exactly n_cities */
    int32_t play_min;         /* R36: playable area h x w uniform in [play_min..H] x [play_min..W]; 0 = H x W */
    int32_t castle_radius;    /* R36: each general has a castle within this many steps (6); 0 = none */
} orc_config;

/* all arrays host memory, game-major; S = plane stride = round_up(H*W, 16) */
typedef struct {
    int16_t *army;            /* [N][S] */
    int8_t *owner;            /* [N][S]  -1 neutral, 0..P-1 */
    int8_t *terrain;          /* [N][S]  0 plain 1 mountain 2 city 3 general */
    int32_t *turn;            /* [N] */
    uint32_t *episode;        /* [N] */
    uint8_t *alive;           /* [N] bit p = player p's general lives */
    int16_t *general_cell;    /* [N][P]  -1 once captured */
    int32_t *land;            /* [N][P] */
    int32_t *army_total;      /* [N][P] */
    int8_t *reward;           /* [N][P] */
    uint8_t *done;            /* [N] bit0 terminated, bit1 truncated */
    int8_t *winner;           /* [N] winning team or -1 */
    int16_t *obs_army;        /* [N][P][S] */
    int8_t *obs_owner;        /* [N][P][S] */
    int8_t *obs_terrain;      /* [N][P][S] */
    uint8_t *obs_vis;         /* [N][P][S] */
    uint32_t *episodes_done;  /* [N] */
    uint32_t *wins;           /* [N][P] */
    uint32_t *truncations;    /* [N] */
    uint32_t *sat_events;     /* [N] */
    uint64_t *obs_digest;     /* [N] or NULL */
    uint8_t *obs_packed;      /* [N][P][S] or NULL: owner, terrain and visibility in one byte (R33) */
    int32_t *score_hist;      /* [N][512][2P] or NULL: ring of the public scoreboard per turn (R34) */
    int8_t *play_size;        /* [N][2] or NULL: playable rows, columns of the current map (R36; R35 padded border) */
    uint32_t *invalid_actions; /* [N] or NULL: diagnostic: actions since reset that were no pass and were not
                                  applied -- index out of range, not the mover's cell, army < 2, target a mountain or off
                                  the board, also when an earlier mover of the same turn made them so (R7) */
} orc_buffers;

/* ------------------------------------------------------------------ Philox
 * Philox4x32-10 (Salmon et al., SC'11): 10 rounds of
 *   (c0,c1,c2,c3) <- (hi(M1*c2)^c1^k0, lo(M1*c2), hi(M0*c0)^c3^k1, lo(M0*c0))
 * with the key bumped by the Weyl constants between rounds. */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* One draw of the stream table (R24/R30):
 * key = seed, counter = (c0, global game id, c2, domain<<24 | player). */
static void draw(const orc_config *cfg, uint32_t gid, uint32_t domain, uint32_t c0,
                 uint32_t c2, uint32_t player, uint32_t w[4])
{
    uint32_t ctr[4] = { c0, gid, c2, (domain << 24) | player };
    uint32_t key[2] = { (uint32_t)(cfg->seed & 0xffffffffu), (uint32_t)(cfg->seed >> 32) };
    orc_philox4x32_10(ctr, key, w);
}

/* floor(u * n / 2^32): uniform index in [0, n) */
static uint32_t mulhi32(uint32_t u, uint32_t n) { return (uint32_t)(((uint64_t)u * n) >> 32); }

/* splitmix64 finaliser (Steele, Lea, Flood 2014) */
uint64_t orc_mix64(uint64_t z)
{
    z ^= z >> 30; z *= 0xBF58476D1CE4E5B9ull;
    z ^= z >> 27; z *= 0x94D049BB133111EBull;
    z ^= z >> 31;
    return z;
}

/* digest key of cell c: the (c+1)-th output of splitmix64 seeded with 0, forced odd (R28) */
uint64_t orc_digest_key(int32_t c) { return orc_mix64((uint64_t)(c + 1) * 0x9E3779B97F4A7C15ull) | 1ull; }

static int plane_stride(const orc_config *cfg) { return (cfg->height * cfg->width + 15) / 16 * 16; }
int32_t orc_plane_stride(const orc_config *cfg) { return plane_stride(cfg); }

static int team_of(const orc_config *cfg, int p) { return p / (cfg->team_size > 0 ? cfg->team_size : 1); }

static int sat_add(int a, int b, uint32_t *sat_events)
{
    int s = a + b;
    if (s > ARMY_MAX) { s = ARMY_MAX; *sat_events += 1; }   /* R21 */
    return s;
}

static int iabs(int x) { return x < 0 ? -x : x; }

/* ------------------------------------------------------------ a1: generator
 * P:L79 gives only the distribution; the algorithm is reading R30, on the
 * synthetic recipe of BASELINE.json (Bernoulli mountains, fixed city count,
 * Manhattan spawn distance, R29). */
static void generate_official(const orc_config *cfg, const orc_buffers *b, int g);
static void generate(const orc_config *cfg, const orc_buffers *b, int g)
{
    if (cfg->map_mode == 1) { generate_official(cfg, b, g); return; }
    const int H = cfg->height, W = cfg->width, P = cfg->n_players, HW = H * W, S = plane_stride(cfg);
    const uint32_t gid = cfg->game_id_base + (uint32_t)g, ep = b->episode[g];
    int16_t *army = b->army + (size_t)g * S;
    int8_t *owner = b->owner + (size_t)g * S, *terrain = b->terrain + (size_t)g * S;
    int16_t *gen = b->general_cell + (size_t)g * P;
    uint32_t w[4];

    for (int c = 0; c < S; ++c) {
        army[c] = 0; owner[c] = OWNER_NEUTRAL;
        terrain[c] = (c < HW) ? T_PLAIN : T_MOUNTAIN;      /* stride padding reads as mountain */
    }

    /* (1) spawn distance window */
    int lo = cfg->spawn_dmin, hi = cfg->spawn_dmax > 0 ? cfg->spawn_dmax : 64;
    if (cfg->spawn_exact) {
        draw(cfg, gid, DOM_SPAWN, 0, ep, 0, w);
        lo = hi = cfg->spawn_dmin + (int)mulhi32(w[1], (uint32_t)(cfg->spawn_dmax - cfg->spawn_dmin + 1));
    }
    /* (2) generals, one after the other */
    int *list = (int *)malloc(sizeof(int) * (size_t)HW);
    for (int p = 0; p < P; ++p) {
        draw(cfg, gid, DOM_SPAWN, (uint32_t)p, ep, 0, w);
        int cell;
        if (p == 0) {
            cell = (int)mulhi32(w[0], (uint32_t)HW);
        } else {
            int l = lo, h = hi, n = 0;
            for (;;) {
                n = 0;
                for (int c = 0; c < HW; ++c) {
                    int mind = 1 << 20, is_general = 0;
                    for (int q = 0; q < p; ++q) {
                        int d = iabs(c / W - gen[q] / W) + iabs(c % W - gen[q] % W);
                        if (d < mind) mind = d;
                        if (c == gen[q]) is_general = 1;
                    }
                    if (!is_general && mind >= l && mind <= h) list[n++] = c;
                }
                if (n > 0) break;
                if (l > 0) l -= 1;          /* infeasible window: widen it by one on each side */
                h += 1;
            }
            cell = list[mulhi32(w[0], (uint32_t)n)];
        }
        gen[p] = (int16_t)cell;
        terrain[cell] = T_GENERAL; owner[cell] = (int8_t)p; army[cell] = 1;   /* R13 */
    }
    /* (3) mountains: one Philox call covers 4 consecutive cells */
    for (int c = 0; c < HW; ++c) {
        if (terrain[c] == T_GENERAL) continue;
        draw(cfg, gid, DOM_MOUNTAIN, (uint32_t)(c >> 2), ep, 0, w);
        if (w[c & 3] < cfg->mountain_thr) terrain[c] = T_MOUNTAIN;
    }
    /* (4) cities, one at a time, uniform over the remaining plain cells (R14) */
    for (int k = 0; k < cfg->n_cities; ++k) {
        int n = 0;
        for (int c = 0; c < HW; ++c) if (terrain[c] == T_PLAIN) list[n++] = c;
        if (n == 0) break;
        draw(cfg, gid, DOM_CITY, (uint32_t)k, ep, 0, w);
        int cell = list[mulhi32(w[0], (uint32_t)n)];
        terrain[cell] = T_CITY;
        army[cell] = (int16_t)(cfg->city_army_lo +
                               (int)mulhi32(w[1], (uint32_t)(cfg->city_army_hi - cfg->city_army_lo + 1)));
    }
    free(list);
    if (b->play_size) { b->play_size[2 * g] = (int8_t)H; b->play_size[2 * g + 1] = (int8_t)W; }
    b->turn[g] = 0;
    b->alive[g] = (uint8_t)((1u << P) - 1u);
}

/* ------------------------------------------------------------ NEXT-3: the official generator (R36)
 * "fills a random 20% of cells with mountains and places 9-11 neutral castles, each pre-loaded with 40-50
 * neutral units.  The two generals are placed at least 17 steps apart, and each player is guaranteed at least one
 * neutral castle within radius 6 of their general"; the distance is the BFS distance; "cells
 * outside the playable area are padded with mountain tokens".  The paper gives the constraints, not the
 * procedure; reading R36 is rejection sampling over whole maps, 1v1 only.  Attempt a = 0..15, every
 * draw of attempt a carries a in the counter's player byte:
 *   (0) one draw fixes the playable size h x w, the spawn window [lo, hi] (in steps) and the castle count;
 *   (1) cells outside the playable rectangle (top-left anchored) are MOUNTAIN; inside, Bernoulli(mountain_thr)
 *       with the same word assignment as R30; on the last attempt the playable area has no mountains;
 *   (2) general 0 uniform over the PLAIN cells (row-major list); none => next attempt;
 *   (3) dist0 = BFS steps from general 0 over non-mountain cells (4-neighbourhood);
 *   (4) general 1 uniform over the PLAIN cells with lo <= dist0 <= hi; none => next attempt (last attempt: widen
 *       the window by one on each side until some cell qualifies, as R30 does);
 *   (5) castle 0 uniform over PLAIN cells with dist0 <= radius, castle 1 over PLAIN cells with dist1 <= radius
 *       (BFS from general 1); none => next attempt (last attempt: over all PLAIN cells); castles 2.. uniform over
 *       the remaining PLAIN cells; garrison lo + mulhi32(u, span) as R14.  radius 0: every castle uniform.
 * Unreachable cells have no distance and never qualify, so an accepted map always connects the two generals. */
enum { MAP_ATTEMPTS = 16, DIST_NONE = 1 << 20 };

static void bfs_steps(const int8_t *terrain, int H, int W, int src, int *dist, int *queue)
{
    for (int c = 0; c < H * W; ++c) dist[c] = DIST_NONE;
    int head = 0, tail = 0;
    dist[src] = 0; queue[tail++] = src;
    while (head < tail) {
        const int c = queue[head++], r = c / W, col = c % W;
        const int nb[4] = { r > 0 ? c - W : -1, r < H - 1 ? c + W : -1, col > 0 ? c - 1 : -1, col < W - 1 ? c + 1 : -1 };
        for (int k = 0; k < 4; ++k) {
            const int n = nb[k];
            if (n < 0 || terrain[n] == T_MOUNTAIN || dist[n] != DIST_NONE) continue;
            dist[n] = dist[c] + 1; queue[tail++] = n;
        }
    }
}

static void generate_official(const orc_config *cfg, const orc_buffers *b, int g)
{
    const int H = cfg->height, W = cfg->width, HW = H * W, S = plane_stride(cfg);
    const uint32_t gid = cfg->game_id_base + (uint32_t)g, ep = b->episode[g];
    int16_t *army = b->army + (size_t)g * S;
    int8_t *owner = b->owner + (size_t)g * S, *terrain = b->terrain + (size_t)g * S;
    int16_t *gen = b->general_cell + (size_t)g * 2;
    int *list = (int *)malloc(sizeof(int) * (size_t)HW * 4);
    int *dist0 = list + HW, *dist1 = list + 2 * HW, *queue = list + 3 * HW;
    uint32_t w[4];

    for (uint32_t a = 0; a < MAP_ATTEMPTS; ++a) {
        const int last = (a == MAP_ATTEMPTS - 1);
        /* (0) sizes of this attempt */
        draw(cfg, gid, DOM_SPAWN, 0, ep, a, w);
        int h = H, wd = W;
        if (cfg->play_min > 0) {
            const int hmin = cfg->play_min < H ? cfg->play_min : H, wmin = cfg->play_min < W ? cfg->play_min : W;
            h = hmin + (int)mulhi32(w[0], (uint32_t)(H - hmin + 1));
            wd = wmin + (int)mulhi32(w[1], (uint32_t)(W - wmin + 1));
        }
        int lo = cfg->spawn_dmin, hi = cfg->spawn_dmax > 0 ? cfg->spawn_dmax : DIST_NONE - 1;
        if (cfg->spawn_exact)
            lo = hi = cfg->spawn_dmin + (int)mulhi32(w[2], (uint32_t)(cfg->spawn_dmax - cfg->spawn_dmin + 1));
        int n_castles = cfg->n_cities;
        if (cfg->n_cities_max > cfg->n_cities)
            n_castles += (int)mulhi32(w[3], (uint32_t)(cfg->n_cities_max - cfg->n_cities + 1));
        /* (1) terrain */
        for (int c = 0; c < S; ++c) { army[c] = 0; owner[c] = OWNER_NEUTRAL; terrain[c] = T_MOUNTAIN; }
        for (int c = 0; c < HW; ++c) {
            if (c / W >= h || c % W >= wd) continue;
            uint32_t m[4];
            draw(cfg, gid, DOM_MOUNTAIN, (uint32_t)(c >> 2), ep, a, m);
            terrain[c] = (!last && m[c & 3] < cfg->mountain_thr) ? T_MOUNTAIN : T_PLAIN;
        }
        /* (2) general 0 */
        draw(cfg, gid, DOM_SPAWN, 1, ep, a, w);
        int n = 0;
        for (int c = 0; c < HW; ++c) if (terrain[c] == T_PLAIN) list[n++] = c;
        if (n == 0) continue;
        const int g0 = list[mulhi32(w[0], (uint32_t)n)];
        /* (3), (4) general 1 at lo..hi steps */
        bfs_steps(terrain, H, W, g0, dist0, queue);
        for (;;) {
            n = 0;
            for (int c = 0; c < HW; ++c)
                if (terrain[c] == T_PLAIN && c != g0 && dist0[c] >= lo && dist0[c] <= hi) list[n++] = c;
            if (n > 0 || !last) break;
            if (lo == 0 && hi >= HW) break;                 /* a one-cell playable area: nothing to place */
            if (lo > 0) lo -= 1;
            hi += 1;
        }
        if (n == 0) continue;
        const int g1 = list[mulhi32(w[1], (uint32_t)n)];
        bfs_steps(terrain, H, W, g1, dist1, queue);
        terrain[g0] = T_GENERAL; owner[g0] = 0; army[g0] = 1;       /* R13 */
        terrain[g1] = T_GENERAL; owner[g1] = 1; army[g1] = 1;
        /* (5) castles */
        int ok = 1;
        for (int k = 0; k < n_castles; ++k) {
            const int *near = (cfg->castle_radius > 0 && k < 2) ? (k == 0 ? dist0 : dist1) : NULL;
            n = 0;
            if (near)
                for (int c = 0; c < HW; ++c) if (terrain[c] == T_PLAIN && near[c] <= cfg->castle_radius) list[n++] = c;
            if (near && n == 0 && !last) { ok = 0; break; }
            if (n == 0)
                for (int c = 0; c < HW; ++c) if (terrain[c] == T_PLAIN) list[n++] = c;
            if (n == 0) break;
            draw(cfg, gid, DOM_CITY, (uint32_t)k, ep, a, w);
            const int cell = list[mulhi32(w[0], (uint32_t)n)];
            terrain[cell] = T_CITY;
            army[cell] = (int16_t)(cfg->city_army_lo +
                                   (int)mulhi32(w[1], (uint32_t)(cfg->city_army_hi - cfg->city_army_lo + 1)));
        }
        if (!ok) continue;
        gen[0] = (int16_t)g0; gen[1] = (int16_t)g1;
        if (b->play_size) { b->play_size[2 * g] = (int8_t)h; b->play_size[2 * g + 1] = (int8_t)wd; }
        break;
    }
    free(list);
    b->turn[g] = 0;
    b->alive[g] = 3;
}

/* ------------------------------------------------- a7: scoreboard (R23) */
static void scoreboard(const orc_config *cfg, const orc_buffers *b, int g)
{
    const int P = cfg->n_players, HW = cfg->height * cfg->width, S = plane_stride(cfg);
    const int16_t *army = b->army + (size_t)g * S;
    const int8_t *owner = b->owner + (size_t)g * S;
    for (int p = 0; p < P; ++p) { b->land[g * P + p] = 0; b->army_total[g * P + p] = 0; }
    for (int c = 0; c < HW; ++c)
        if (owner[c] >= 0) { b->land[g * P + owner[c]] += 1; b->army_total[g * P + owner[c]] += army[c]; }
}

/* ------------------------- R34: the raw material of the paper's two temporal
 * tokens, "a 512-step sliding window of the opponent's total army count and a matching window of their total
 * land count".  Slot (turn mod 512) of the game's ring holds (land[p], army_total[p]) of every player as the
 * scoreboard stands at the end of that turn (turn 0: the freshly generated board). */
enum { HIST_LEN = 512 };
static void record_history(const orc_config *cfg, const orc_buffers *b, int g)
{
    const int P = cfg->n_players;
    if (!b->score_hist) return;
    int32_t *slot = b->score_hist + ((size_t)g * HIST_LEN + (size_t)(b->turn[g] % HIST_LEN)) * 2 * P;
    for (int p = 0; p < P; ++p) {
        slot[2 * p] = b->land[g * P + p];
        slot[2 * p + 1] = b->army_total[g * P + p];
    }
}

/* ------------------------- a10 + a11: fog of war and the four planes (R18, R19, R32)
 * A cell is visible to p iff it or one of its 8 Moore neighbours is owned by a member of p's team. */
static void observe(const orc_config *cfg, const orc_buffers *b, int g, size_t obs_game_index)
{
    const int H = cfg->height, W = cfg->width, P = cfg->n_players, HW = H * W, S = plane_stride(cfg);
    const int16_t *army = b->army + (size_t)g * S;
    const int8_t *owner = b->owner + (size_t)g * S, *terrain = b->terrain + (size_t)g * S;
    for (int p = 0; p < P; ++p) {
        size_t o = (obs_game_index * P + p) * (size_t)S;
        for (int c = 0; c < S; ++c) {
            int vis = 0;
            if (c < HW) {
                int r = c / W, col = c % W;
                for (int dr = -1; dr <= 1; ++dr)
                    for (int dc = -1; dc <= 1; ++dc) {
                        int rr = r + dr, cc = col + dc;
                        if (rr < 0 || rr >= H || cc < 0 || cc >= W) continue;
                        int t = owner[rr * W + cc];
                        if (t >= 0 && team_of(cfg, t) == team_of(cfg, p)) vis = 1;
                    }
            }
            b->obs_army[o + c] = vis ? army[c] : 0;
            b->obs_owner[o + c] = vis ? owner[c] : (int8_t)OWNER_FOG;
            b->obs_terrain[o + c] = vis ? terrain[c] : (int8_t)T_FOG;
            b->obs_vis[o + c] = (uint8_t)vis;
            /* R33: the three byte planes in one byte.  Visible: bit 7 set, bits 4-5 the
             * terrain, bits 0-3 owner + 2 (1 = neutral, 2.. = player 0..); fogged: 0. */
            if (b->obs_packed)
                b->obs_packed[o + c] = vis ? (uint8_t)(0x80 | (terrain[c] << 4) | (owner[c] + 2)) : (uint8_t)0;
        }
    }
}

/* ------------------------------------------------------- R28: observation digest
 * h_p = sum_c pack(p,c) * K(c) mod 2^64, chained through mix64 player by player,
 * then the step's reward / done / winner bits. */
static uint64_t chain_digest(const orc_config *cfg, const orc_buffers *b, int g, size_t obs_game_index,
                             uint64_t d)
{
    const int P = cfg->n_players, HW = cfg->height * cfg->width, S = plane_stride(cfg);
    for (int p = 0; p < P; ++p) {
        size_t o = (obs_game_index * P + p) * (size_t)S;
        uint64_t h = 0;
        for (int c = 0; c < HW; ++c) {
            uint64_t pack = (uint64_t)(uint16_t)b->obs_army[o + c]
                          | ((uint64_t)(b->obs_owner[o + c] + 2) << 16)
                          | ((uint64_t)b->obs_terrain[o + c] << 20)
                          | ((uint64_t)b->obs_vis[o + c] << 24);
            h += pack * orc_digest_key(c);
        }
        d = orc_mix64(d ^ h);
    }
    uint64_t tail = (uint64_t)b->done[g] | ((uint64_t)(uint8_t)(b->winner[g] + 2) << 8);
    for (int p = 0; p < P; ++p) tail |= (uint64_t)(b->reward[g * P + p] + 1) << (16 + 2 * p);
    return orc_mix64(d ^ tail);
}

/* -------------------------------------------------------- a2: decode + validate
 * a = cell*9 + k; k = 0 pass, else dir = (k-1)>>1 (0 up,1 down,2 left,3 right), half = (k-1)&1 (R22).
 * Returns 1 and fills src/dst/half iff the move is valid for p on the board as it stands (R5, R10). */
static int decode(const orc_config *cfg, const int16_t *army, const int8_t *owner, const int8_t *terrain,
                  int p, int32_t a, int *src, int *dst, int *half)
{
    const int H = cfg->height, W = cfg->width, HW = H * W;
    if (a < 0 || a >= 9 * HW) return 0;
    int cell = a / 9, k = a % 9;
    if (k == 0) return 0;
    int dir = (k - 1) >> 1;
    int r = cell / W, col = cell % W;
    if (dir == 0) r -= 1; else if (dir == 1) r += 1; else if (dir == 2) col -= 1; else col += 1;
    if (r < 0 || r >= H || col < 0 || col >= W) return 0;
    int t = r * W + col;
    if (owner[cell] != p || army[cell] < 2 || terrain[t] == T_MOUNTAIN) return 0;
    *src = cell; *dst = t; *half = (k - 1) & 1;
    return 1;
}

/* ------------------------------------------------------ a12: valid-action sampler (R24, R25)
 * Valid list in (direction, cell) order; one Philox call per player and step. */
static int32_t sample_action(const orc_config *cfg, const orc_buffers *b, int g, int p, uint32_t global_step)
{
    const int HW = cfg->height * cfg->width, S = plane_stride(cfg);
    const int16_t *army = b->army + (size_t)g * S;
    const int8_t *owner = b->owner + (size_t)g * S, *terrain = b->terrain + (size_t)g * S;
    uint32_t w[4];
    draw(cfg, cfg->game_id_base + (uint32_t)g, DOM_ACTION, 0, global_step, (uint32_t)p, w);
    if (w[0] < cfg->pass_thr) return 0;
    int32_t *list = (int32_t *)malloc(sizeof(int32_t) * 4 * (size_t)HW);
    int n = 0, s, d, h;
    for (int dir = 0; dir < 4; ++dir)
        for (int c = 0; c < HW; ++c) {
            int32_t a = c * 9 + 1 + 2 * dir;
            if (decode(cfg, army, owner, terrain, p, a, &s, &d, &h)) list[n++] = a;
        }
    int32_t action = 0;
    if (n > 0) {
        if (w[3] < cfg->bias_thr) {                    /* R25: largest owned stack, ties -> lowest cell */
            int best = -1;
            for (int c = 0; c < HW; ++c)
                if (owner[c] == p && (best < 0 || army[c] > army[best])) best = c;
            int nb = 0; int32_t blist[4];
            for (int dir = 0; best >= 0 && dir < 4; ++dir) {
                int32_t a = best * 9 + 1 + 2 * dir;
                if (decode(cfg, army, owner, terrain, p, a, &s, &d, &h)) blist[nb++] = a;
            }
            if (nb > 0) { n = nb; for (int i = 0; i < nb; ++i) list[i] = blist[i]; }
        }
        action = list[mulhi32(w[1], (uint32_t)n)] + (w[2] < cfg->half_thr ? 1 : 0);
    }
    free(list);
    return action;
}

/* a4: general capture (R11) */
static void capture(const orc_config *cfg, const orc_buffers *b, int g, int p, int q, int dst)
{
    const int HW = cfg->height * cfg->width, S = plane_stride(cfg), P = cfg->n_players;
    int16_t *army = b->army + (size_t)g * S;
    int8_t *owner = b->owner + (size_t)g * S, *terrain = b->terrain + (size_t)g * S;
    b->alive[g] &= (uint8_t)~(1u << q);
    b->general_cell[g * P + q] = -1;
    terrain[dst] = T_CITY;
    for (int c = 0; c < HW; ++c)
        if (owner[c] == q) {
            owner[c] = (int8_t)p;
            army[c] = (cfg->rule_flags & RULE_CAPTURE_HALF_FLOOR) ? (int16_t)(army[c] >> 1)
                                                                   : (int16_t)((army[c] + 1) >> 1);
        }
}

/* ------------------------------------------------------------------ one game, one turn
 * SURVEY/DESIGN step(game, actions[P]) in the paper's order: moves, growth,
 * scoreboard, termination + reward, auto-reset, observation. */
static void step_game(const orc_config *cfg, const orc_buffers *b, int g, const int32_t *actions,
                      size_t obs_game_index)
{
    const int P = cfg->n_players, HW = cfg->height * cfg->width, S = plane_stride(cfg);
    int16_t *army = b->army + (size_t)g * S;
    int8_t *owner = b->owner + (size_t)g * S, *terrain = b->terrain + (size_t)g * S;

    if (!cfg->auto_reset && b->done[g] != 0) {            /* R31: frozen */
        for (int p = 0; p < P; ++p) b->reward[g * P + p] = 0;
        observe(cfg, b, g, obs_game_index);
        return;
    }
    /* 1. moves, sequentially, each re-validated on the current board (R6, R7) */
    int first = (cfg->rule_flags & RULE_ROTATE_PRIORITY) ? b->turn[g] % P : 0;
    for (int i = 0; i < P; ++i) {
        int p = (first + i) % P, src, dst, half;
        if (!decode(cfg, army, owner, terrain, p, actions[p], &src, &dst, &half)) {
            const int32_t a = actions[p];
            const int is_pass = a >= 0 && a < 9 * HW && a % 9 == 0;          /* R22: k = 0 */
            if (!is_pass && b->invalid_actions) b->invalid_actions[g] += 1;   /* an invalid action is a pass (R5, R10) */
            continue;
        }
        int m = half ? army[src] / 2 : army[src] - 1;     /* R4 */
        army[src] = (int16_t)(army[src] - m);
        int t = owner[dst], d = army[dst];
        if (t == p) {
            army[dst] = (int16_t)sat_add(d, m, &b->sat_events[g]);                      /* R8 */
        } else if (t >= 0 && team_of(cfg, t) == team_of(cfg, p)) {                      /* P:L97, R19 */
            army[dst] = (int16_t)sat_add(d, m, &b->sat_events[g]);
            if (terrain[dst] != T_GENERAL) owner[dst] = (int8_t)p;
        } else if (m > d) {
            army[dst] = (int16_t)(m - d);
            owner[dst] = (int8_t)p;
            if (terrain[dst] == T_GENERAL && t >= 0) capture(cfg, b, g, p, t, dst);     /* R11, R12 */
        } else {
            army[dst] = (int16_t)(d - m);                 /* tie -> 0, previous owner keeps the cell */
        }
    }
    /* 2. turn counter, then growth (R1, R2, R3) */
    b->turn[g] += 1;
    if (b->turn[g] % 2 == 0)
        for (int c = 0; c < HW; ++c)
            if (owner[c] >= 0 && (terrain[c] == T_CITY || terrain[c] == T_GENERAL))
                army[c] = (int16_t)sat_add(army[c], 1, &b->sat_events[g]);
    if (b->turn[g] % 50 == 0)
        for (int c = 0; c < HW; ++c) {
            if (owner[c] < 0) continue;
            if ((cfg->rule_flags & RULE_TICK_PLAIN_ONLY) && terrain[c] != T_PLAIN) continue;
            army[c] = (int16_t)sat_add(army[c], 1, &b->sat_events[g]);
        }
    /* 3. scoreboard */
    scoreboard(cfg, b, g);
    /* 4. termination, reward, done (R16, R20) */
    int n_teams = (P + cfg->team_size - 1) / cfg->team_size, living = 0, last = -1;
    for (int t = 0; t < n_teams; ++t) {
        int any = 0;
        for (int p = 0; p < P; ++p) if (team_of(cfg, p) == t && ((b->alive[g] >> p) & 1)) any = 1;
        if (any) { living += 1; last = t; }
    }
    int terminated = living <= 1;
    int truncated = !terminated && cfg->max_turns > 0 && b->turn[g] >= cfg->max_turns;
    b->done[g] = (uint8_t)((terminated ? DONE_TERMINATED : 0) | (truncated ? DONE_TRUNCATED : 0));
    b->winner[g] = (int8_t)(terminated ? last : -1);
    for (int p = 0; p < P; ++p) {
        int8_t r = 0;
        if (terminated) r = (team_of(cfg, p) == last) ? 1 : -1;
        b->reward[g * P + p] = r;
        if (r > 0) b->wins[g * P + p] += 1;
    }
    if (b->done[g]) b->episodes_done[g] += 1;
    if (truncated) b->truncations[g] += 1;
    /* 5. auto-reset (R17): reward/done describe the finished episode, state + obs the new one */
    if (b->done[g] && cfg->auto_reset) {
        b->episode[g] += 1;
        generate(cfg, b, g);
        scoreboard(cfg, b, g);
    }
    record_history(cfg, b, g);                                /* R34: the scoreboard as this call leaves it */
    /* 6. observation of the state at the end of the call (R32) */
    observe(cfg, b, g, obs_game_index);
}

/* ===================================================================== C ABI (ctypes) */
int32_t orc_reset(const orc_config *cfg, const orc_buffers *b)
{
    const int P = cfg->n_players;
    for (int g = 0; g < cfg->n_games; ++g) {
        b->episode[g] = 0;
        generate(cfg, b, g);
        scoreboard(cfg, b, g);
        b->done[g] = 0; b->winner[g] = -1;
        b->episodes_done[g] = 0; b->truncations[g] = 0; b->sat_events[g] = 0;
        if (b->invalid_actions) b->invalid_actions[g] = 0;
        for (int p = 0; p < P; ++p) { b->reward[g * P + p] = 0; b->wins[g * P + p] = 0; }
        record_history(cfg, b, g);
        observe(cfg, b, g, (size_t)g);
        if (b->obs_digest) b->obs_digest[g] = chain_digest(cfg, b, g, (size_t)g, 0);
    }
    return 0;
}

/* the sampler alone: actions_out[N][P] drawn on the board as it stands */
int32_t orc_sample(const orc_config *cfg, const orc_buffers *b, uint32_t global_step, int32_t *actions_out)
{
    const int P = cfg->n_players;
    for (int g = 0; g < cfg->n_games; ++g)
        for (int p = 0; p < P; ++p) {
            int frozen = !cfg->auto_reset && b->done[g] != 0;
            actions_out[g * P + p] = frozen ? 0 : sample_action(cfg, b, g, p, global_step);
        }
    return 0;
}

/* one turn for all games; actions == NULL -> all P players' actions are drawn first, on the
 * pre-move board (players choose without seeing each other's move), then applied */
int32_t orc_step(const orc_config *cfg, const orc_buffers *b, const int32_t *actions, uint32_t global_step,
                 int32_t *actions_out)
{
    const int P = cfg->n_players;
    int32_t a[8];
    for (int g = 0; g < cfg->n_games; ++g) {
        int frozen = !cfg->auto_reset && b->done[g] != 0;
        for (int p = 0; p < P; ++p) {
            /* R31: a frozen game applies nothing, whatever the caller passed; actions_out reports the action
             * actually applied (include/generals.h), i.e. 0 = pass */
            a[p] = frozen ? 0 : (actions ? actions[g * P + p] : sample_action(cfg, b, g, p, global_step));
            if (actions_out) actions_out[g * P + p] = a[p];
        }
        step_game(cfg, b, g, a, (size_t)g);
        if (b->obs_digest && !frozen) b->obs_digest[g] = chain_digest(cfg, b, g, (size_t)g, b->obs_digest[g]);
    }
    return 0;
}

/* K sampled turns. obs_mode ORC_OBS_EVERY_STEP: step k's planes / reward / done / winner land in
 * slot k of K-times-larger buffers; otherwise only the last step's are kept (slot 0). */
int32_t orc_rollout(const orc_config *cfg, const orc_buffers *b, int32_t K, uint32_t global_step0,
                    int32_t obs_mode)
{
    const int N = cfg->n_games, P = cfg->n_players;
    if (obs_mode != ORC_OBS_EVERY_STEP) {
        for (int k = 0; k < K; ++k) orc_step(cfg, b, NULL, global_step0 + (uint32_t)k, NULL);
        return 0;
    }
    const size_t S = (size_t)plane_stride(cfg);
    for (int k = 0; k < K; ++k) {
        orc_buffers v = *b;
        v.obs_army += (size_t)k * N * P * S; v.obs_owner += (size_t)k * N * P * S;
        v.obs_terrain += (size_t)k * N * P * S; v.obs_vis += (size_t)k * N * P * S;
        if (v.obs_packed) v.obs_packed += (size_t)k * N * P * S;
        v.reward += (size_t)k * N * P; v.done += (size_t)k * N; v.winner += (size_t)k * N;
        if (k > 0) {                                           /* carry the frozen game's flags forward */
            memcpy(v.done, v.done - N, (size_t)N);
            memcpy(v.winner, v.winner - N, (size_t)N);
        }
        orc_step(cfg, &v, NULL, global_step0 + (uint32_t)k, NULL);
    }
    return 0;
}

/* observation + scoreboard of a hand-built state (tests) */
/* The entry point for states written by the caller (hand-built boards).  R40: in every state the rules
 * produce, the GENERAL cells are exactly the cells general_cell[p] of their owners -- both generators place them so,
 * and a captured general becomes a CITY (R11).  PAPER.md speaks of "unclaimed castles/generals" once (Table IV ch. 3,
 * P:L361) and gives no rule for an unclaimed general; a GENERAL cell that is nobody's recorded general is therefore
 * turned into a CITY here (it is a structure that nobody's elimination hangs on), so that step_game never meets one. */
int32_t orc_observe(const orc_config *cfg, const orc_buffers *b)
{
    const int P = cfg->n_players, HW = cfg->height * cfg->width, S = plane_stride(cfg);
    for (int g = 0; g < cfg->n_games; ++g) {
        int8_t *owner = b->owner + (size_t)g * S, *terrain = b->terrain + (size_t)g * S;
        for (int c = 0; c < HW; ++c)
            if (terrain[c] == T_GENERAL && (owner[c] < 0 || owner[c] >= P || b->general_cell[g * P + owner[c]] != c))
                terrain[c] = T_CITY;
        scoreboard(cfg, b, g);
        observe(cfg, b, g, (size_t)g);
    }
    return 0;
}

/* ===================================================================== NEXT-1: the 38-channel feature tensor
 * PAPER.md Appendix A and Table IV.  One call per turn and game: it folds the current
 * observation into the per-episode memory and writes, for each player p as the agent, C = 24 + 2 * 7 = 38 float
 * maps feat[g][p][ch][S] (more than two players: reading R38 below).  Readings (DESIGN.md
 * R35): the memory is cleared when turn == 0 (a new episode always starts there); "opponent army (last observed)"
 * is the public scoreboard; channel 9 counts every visible neutral-owned cell; channel 21 is 0 where the enemy was
 * never seen or is visible now; deltas that reach before the episode's first frame are 0; coordinates are
 * col / (W - 1) and row / (H - 1); stride padding cells are 0 in every channel; the padded border of a smaller
 * playable area (play_size) is a known mountain from turn 0. */
enum { FEAT_C = 38, FEAT_HIST = 7, FEAT_RING = 8 };

typedef struct {
    uint8_t *bits;        /* [N][P][5][S]  seen, enemy_seen, generals, castles, mountains (0 / 1) */
    int16_t *last_army;   /* [N][P][S]     enemy army last observed on the cell */
    int32_t *last_turn;   /* [N][P][S]     turn of that observation, -1 = never */
    int16_t *hist;        /* [N][P][2][8][S]  own_army / enemy_army frames, slot turn mod 8 */
} orc_feat_state;

#include <math.h>

int32_t orc_features(const orc_config *cfg, const orc_buffers *b, const orc_feat_state *m, float *feat)
{
    const int H = cfg->height, W = cfg->width, P = cfg->n_players, HW = H * W, S = plane_stride(cfg);
    /* More than two players (R38; "the same observation ... interface for the 1v1, 2v2, and free-for-all
     * formats"): "the agent" is player p, "the opponent" is every player who is not on p's team; visibility is the
     * team's (R19); an ally's cells are visible but neither own, enemy nor neutral; the opponent's scoreboard
     * entries (ch 18, 19) are the sums over all enemies.  With two players this is Table IV verbatim. */
    for (int g = 0; g < cfg->n_games; ++g) {
        const int16_t *army = b->army + (size_t)g * S;
        const int8_t *owner = b->owner + (size_t)g * S, *terrain = b->terrain + (size_t)g * S;
        const int t = b->turn[g];
        for (int p = 0; p < P; ++p) {
            const int team = team_of(cfg, p);
            int opp_land = 0, opp_army = 0;
            for (int q = 0; q < P; ++q)
                if (team_of(cfg, q) != team) { opp_land += b->land[g * P + q]; opp_army += b->army_total[g * P + q]; }
            const size_t gp = (size_t)g * P + p;
            uint8_t *bits = m->bits + gp * 5 * S;
            int16_t *last_army = m->last_army + gp * S;
            int32_t *last_turn = m->last_turn + gp * S;
            int16_t *hist_own = m->hist + (gp * 2 + 0) * FEAT_RING * S, *hist_en = m->hist + (gp * 2 + 1) * FEAT_RING * S;
            float *out = feat + gp * FEAT_C * S;
            if (t == 0) {                                      /* new episode: forget */
                memset(bits, 0, (size_t)5 * S);
                memset(last_army, 0, sizeof(int16_t) * S);
                for (int c = 0; c < S; ++c) last_turn[c] = -1;
                memset(hist_own, 0, sizeof(int16_t) * FEAT_RING * S);
                memset(hist_en, 0, sizeof(int16_t) * FEAT_RING * S);
            }
            memset(out, 0, sizeof(float) * FEAT_C * S);
            /* Table IV ch 8 "visible mountains U known padded border", ch 13 "... or unseen padded border": with a
             * playable area smaller than the board (R36) the cells outside it are mountains the agent knows of
             * from the first turn */
            /* (0 = not recorded, e.g. a board written by hand: the full board) */
            const int ph = (b->play_size && b->play_size[2 * g] > 0) ? b->play_size[2 * g] : H;
            const int pw = (b->play_size && b->play_size[2 * g + 1] > 0) ? b->play_size[2 * g + 1] : W;
            for (int c = 0; c < HW; ++c) {
                const int r = c / W, col = c % W;
                if (r >= ph || col >= pw) bits[4 * S + c] = 1;
                int vis = 0;                                   /* own cells and their 8 neighbours */
                for (int dr = -1; dr <= 1; ++dr)
                    for (int dc = -1; dc <= 1; ++dc) {
                        int rr = r + dr, cc = col + dc;
                        if (rr >= 0 && rr < H && cc >= 0 && cc < W && owner[rr * W + cc] >= 0 &&
                            team_of(cfg, owner[rr * W + cc]) == team) vis = 1;
                    }
                const int a = army[c], o = owner[c], tr = terrain[c];
                const int own_a = (o == p) ? a : 0;
                const int en_vis = vis && o >= 0 && team_of(cfg, o) != team;
                const int en_a = en_vis ? a : 0;
                /* fold into the memory */
                bits[0 * S + c] |= (uint8_t)vis;
                bits[1 * S + c] |= (uint8_t)en_vis;
                bits[2 * S + c] |= (uint8_t)(vis && tr == T_GENERAL);
                bits[3 * S + c] |= (uint8_t)(vis && tr == T_CITY);
                bits[4 * S + c] |= (uint8_t)(vis && tr == T_MOUNTAIN);
                if (en_vis) { last_army[c] = (int16_t)a; last_turn[c] = t; }
                hist_own[(t % FEAT_RING) * S + c] = (int16_t)own_a;
                hist_en[(t % FEAT_RING) * S + c] = (int16_t)en_a;
                /* Table IV */
                out[0 * S + c] = (float)(vis ? a : 0);
                out[1 * S + c] = (float)own_a;
                out[2 * S + c] = (float)en_a;
                out[3 * S + c] = (float)((vis && o == OWNER_NEUTRAL) ? a : 0);
                for (int k = 0; k < 5; ++k) out[(4 + k) * S + c] = (float)bits[k * S + c];
                out[9 * S + c] = (float)(vis && o == OWNER_NEUTRAL);
                out[10 * S + c] = (float)(o == p);
                out[11 * S + c] = (float)en_vis;
                out[12 * S + c] = (float)(!vis);
                out[13 * S + c] = (float)(!vis && (bits[2 * S + c] | bits[3 * S + c] | bits[4 * S + c]));
                out[14 * S + c] = (float)t;
                out[15 * S + c] = (float)(t % 50) / 50.0f;
                out[16 * S + c] = (float)b->land[g * P + p];
                out[17 * S + c] = (float)b->army_total[g * P + p];
                out[18 * S + c] = (float)opp_land;
                out[19 * S + c] = (float)opp_army;
                out[20 * S + c] = (float)last_army[c];
                out[21 * S + c] = (last_turn[c] < 0 || en_vis) ? 0.0f : logf(1.0f + (float)(t - last_turn[c])) / 5.0f;
                out[22 * S + c] = W > 1 ? (float)col / (float)(W - 1) : 0.0f;
                out[23 * S + c] = H > 1 ? (float)r / (float)(H - 1) : 0.0f;
                for (int k = 0; k < FEAT_HIST; ++k) {
                    if (t - k - 1 < 0) continue;               /* before the first frame of the episode: 0 */
                    const int s1 = ((t - k) % FEAT_RING) * S + c, s0 = ((t - k - 1) % FEAT_RING) * S + c;
                    out[(24 + k) * S + c] = (float)(hist_own[s1] - hist_own[s0]);
                    out[(31 + k) * S + c] = (float)(hist_en[s1] - hist_en[s0]);
                }
            }
        }
    }
    return 0;
}

/* The same tensor in bfloat16 ("half that in bf16"; DESIGN R37): every fp32 value of orc_features
 * rounded to the nearest bfloat16, ties to even (all values are finite), returned as the 16 bit patterns.  Army counts
 * above 256 are not exact in bfloat16; that is the format's resolution, not a tolerance of the method. */
static uint16_t bf16_rne(float f)
{
    uint32_t u;
    memcpy(&u, &f, sizeof u);
    u += 0x7FFFu + ((u >> 16) & 1u);
    return (uint16_t)(u >> 16);
}

int32_t orc_features_bf16(const orc_config *cfg, const orc_buffers *b, const orc_feat_state *m, float *scratch,
                          uint16_t *feat16)
{
    const int32_t rc = orc_features(cfg, b, m, scratch);
    if (rc != 0) return rc;
    const size_t n = (size_t)cfg->n_games * (size_t)cfg->n_players * FEAT_C * (size_t)plane_stride(cfg);
    for (size_t i = 0; i < n; ++i) feat16[i] = bf16_rne(scratch[i]);
    return 0;
}

/* ===================================================================== NEXT-2: the two temporal tokens' windows
 * PAPER.md P:L141 "Two additional non-spatial tokens carry global temporal statistics ...: a 512-step sliding window
 * of the opponent's total army count and a matching window of their total land count" (also P:L312).  Reading R39
 * (DESIGN.md): for game g and agent p, win[g][p][0][i] is the enemies' summed army total and win[g][p][1][i] their
 * summed land count at turn t - 511 + i of the CURRENT episode (t = turn[g]; i = 511 is the turn the scoreboard
 * stands at now, i = 0 the oldest step of the window), and 0 for the steps before the episode's first turn.
 * "The opponent" is every player off p's team (R38).  The values are read from the ring of R34 (slot turn mod 512). */
int32_t orc_history_windows(const orc_config *cfg, const orc_buffers *b, int32_t *win)
{
    const int P = cfg->n_players;
    if (!b->score_hist) return -1;
    for (int g = 0; g < cfg->n_games; ++g) {
        const int t = b->turn[g];
        for (int p = 0; p < P; ++p) {
            int32_t *army_w = win + (((size_t)g * P + p) * 2 + 0) * HIST_LEN;
            int32_t *land_w = win + (((size_t)g * P + p) * 2 + 1) * HIST_LEN;
            for (int i = 0; i < HIST_LEN; ++i) {
                const int tt = t - (HIST_LEN - 1) + i;            /* the turn this entry of the window shows */
                int32_t army = 0, land = 0;
                if (tt >= 0) {
                    const int32_t *slot = b->score_hist + ((size_t)g * HIST_LEN + (size_t)(tt % HIST_LEN)) * 2 * P;
                    for (int q = 0; q < P; ++q)
                        if (team_of(cfg, q) != team_of(cfg, p)) { land += slot[2 * q]; army += slot[2 * q + 1]; }
                }
                army_w[i] = army;
                land_w[i] = land;
            }
        }
    }
    return 0;
}
