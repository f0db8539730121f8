/*
 * generals.h -- C ABI of the B200-native batched Generals.io environment step.
 *
 * The hot path of arXiv 2606.23348 ("P:Lnn" = line nn of PAPER.md; "Rn" = reading n of DESIGN.md):
 * for N independent games at once, apply every player's move with combat / capture / land transfer
 * (section IV-D/E), army growth (IV-C), termination, reward and auto-reset
 * (P:L61), and emit each player's fog-of-war observation planes (IV-B, IV-G).
 *
 * Conventions for every call below
 *   - All `gen_buffers` members are DEVICE pointers owned by the caller (e.g. torch tensors), 16-byte
 *     aligned, sized as `gen_query_sizes` reports.  The library owns only the `gen_env` handle; it
 *     never allocates board memory, never synchronises and never copies to the host (except
 *     `gen_step_host`, which says so).  A call enqueues kernels on `cuda_stream` (a cudaStream_t
 *     passed as void*, NULL = the legacy default stream) and returns; buffers must stay alive until
 *     that work has completed.
 *   - Return value: 0 = GEN_OK, negative = error (see gen_error_string).  Invalid GAME actions are
 *     not errors: they are passes (R5, R10).
 *   - Layout: plane stride S = round_up(H*W, 16) cells; cell index c = row*W + col.  Encodings (R18):
 *     terrain int8 {0 plain, 1 mountain, 2 city(castle), 3 general}; owner int8 {-1 neutral, 0..P-1};
 *     army int16 >= 0 (saturating at 32767, R21).  Fogged cells read army 0, owner -2, terrain 4.
 *   - Determinism: outputs are a pure function of (config, policy, seed, global game id =
 *     game_id_base + g, actions); independent of N, of launch geometry, and of whether K steps were
 *     made by K gen_step calls or one gen_rollout(K).
 *   - sm_100a only.  There is no CPU fallback and no other architecture.
 */
#ifndef GENERALS_H_
#define GENERALS_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
    GEN_OK = 0,
    GEN_ERR_NULL = -1,    /* a required pointer is NULL */
    GEN_ERR_CONFIG = -2,  /* H/W/P/team_size out of range, lo > hi, infeasible counts */
    GEN_ERR_ALIGN = -3,   /* a device pointer is not 16-byte aligned */
    GEN_ERR_ARG = -4,     /* K <= 0, unknown flag, missing buffer for the requested mode */
    GEN_ERR_CUDA = -5,    /* launch / runtime error (cudaGetLastError captured; see gen_last_cuda_error) */
    GEN_ERR_SIZE = -6     /* gen_step_noalloc: the batch needs more than GEN_NOALLOC_SCRATCH_BYTES of built-in scratch */
};

/* rule_flags: alternative readings of the paper, honoured by both sides (R2, R11, R6) */
enum {
    GEN_RULE_TICK_PLAIN_ONLY = 1,    /* 50-turn tick skips cities and generals */
    GEN_RULE_CAPTURE_HALF_FLOOR = 2, /* transferred armies are floor(a/2) instead of ceil(a/2) */
    GEN_RULE_ROTATE_PRIORITY = 4     /* first mover is turn % P instead of player 0 */
};

/* gen_rollout flags */
enum {
    GEN_OBS_DIGEST = 0,     /* chain a 64-bit digest of every step's observation (R28); write final-step planes */
    GEN_OBS_EVERY_STEP = 1, /* write every step's planes / reward / done / winner to slot k of [K]-strided buffers */
    GEN_OBS_NONE = 2        /* state only (reported separately, never the headline) */
};

/* gen_reset flags */
enum { GEN_KEEP_EPISODE = 1 /* regenerate with the episode counters found in the buffer */ };

typedef struct gen_config {
    int32_t n_games;       /* N >= 0 */
    int32_t height, width; /* 1..32 each, H*W >= 2 */
    int32_t n_players;     /* P, 2..8 */
    int32_t team_size;     /* 1 = 1v1 / free-for-all; teams are p / team_size (R19) */
    int32_t n_cities;      /* neutral castles placed at reset (R14) */
    int32_t city_army_lo, city_army_hi; /* castle garrison uniform in [lo, hi] */
    int32_t spawn_dmin;    /* min Manhattan distance between generals (R29) */
    int32_t spawn_dmax;    /* 0 = unbounded; 1v1 window [dmin, dmax] */
    int32_t spawn_exact;   /* 1: per game draw d ~ U{dmin..dmax} and spawn at exactly d (P:L169 curriculum) */
    int32_t max_turns;     /* 0 = none; truncation (R16) */
    int32_t auto_reset;    /* 1: a finished game is regenerated inside the same call (R17) */
    uint32_t rule_flags;
    uint32_t game_id_base; /* global game id = game_id_base + g keys every random draw */
    uint32_t mountain_thr; /* P(mountain) = mountain_thr / 2^32 per non-general cell */
    uint64_t seed;         /* Philox4x32-10 key */
    /* the official map generator (R36).  All zero = the synthetic
     * generator of R30 (BASELINE configs 1-5). */
    int32_t map_mode;      /* 0 synthetic (R30); 1 official: spawn distance in BFS steps, connected generals, castle
                              guarantee, optional mountain-padded playable area.  1v1 only */
    int32_t n_cities_max;  /* map_mode 1: castle count uniform in [n_cities, n_cities_max] (9-11); 0 = n_cities */
    int32_t play_min;      /* map_mode 1: playable area h x w uniform in [play_min, H] x [play_min, W], top-left
                              anchored, the rest mountains; 0 = the full board */
    int32_t castle_radius; /* map_mode 1: each general has a castle within this many steps (6); 0 = no guarantee */
} gen_config;

/* probabilities as uint32 thresholds floor(p * 2^32): no float enters the hot path (R24, R25) */
typedef struct gen_policy {
    uint32_t pass_thr; /* P(pass) */
    uint32_t half_thr; /* P(half split | move) */
    uint32_t bias_thr; /* P(restrict to the largest owned stack) */
} gen_policy;

/* Device buffers.  [N] etc. are element counts; S = plane stride; K = slots of an EVERY_STEP rollout
 * (1 otherwise).  "state" members are read and written; "out" members are written only. */
typedef struct gen_buffers {
    int16_t *army;           /* state [N][S] */
    int8_t *owner;           /* state [N][S] */
    int8_t *terrain;         /* state [N][S] */
    int32_t *turn;           /* state [N] */
    uint32_t *episode;       /* state [N] */
    uint8_t *alive;          /* state [N]   bit p = player p's general lives */
    int16_t *general_cell;   /* state [N][P]  -1 once captured */
    int32_t *land;           /* state [N][P]  public scoreboard (R23) */
    int32_t *army_total;     /* state [N][P] */
    int8_t *reward;          /* out   [K][N][P]  +1 / -1 on the terminal step, else 0 (R20) */
    uint8_t *done;           /* state [K][N]  bit0 terminated, bit1 truncated */
    int8_t *winner;          /* state [K][N]  winning team or -1 */
    int16_t *obs_army;       /* out   [K][N][P][S] */
    int8_t *obs_owner;       /* out   [K][N][P][S] */
    int8_t *obs_terrain;     /* out   [K][N][P][S] */
    uint8_t *obs_vis;        /* out   [K][N][P][S] */
    uint32_t *episodes_done; /* state [N]   accumulators */
    uint32_t *wins;          /* state [N][P] */
    uint32_t *truncations;   /* state [N] */
    uint32_t *sat_events;    /* state [N]   int16 saturations (R21) */
    uint64_t *obs_digest;    /* state [N]   may be NULL for gen_reset / gen_step (no digest then) */
    int32_t *actions_out;    /* out   [K][N][P]  the actions actually applied; may be NULL */
    uint32_t *bitboards;     /* state [N][P+3][BW]  derived cache, may be NULL (see below) */
    uint8_t *obs_packed;     /* out   [K][N][P][S]  packed observation, may be NULL (see below) */
    int32_t *score_hist;     /* state [N][512][2P]  scoreboard history ring, may be NULL (see below) */
    uint32_t *step_epoch;    /* state [2][ceil(N/4)]  launch chaining of gen_step, may be NULL (see below); zeroed once */
    int8_t *play_size;       /* state [N][2]  playable rows, columns of the current map, may be NULL: written by the
                                generators (H, W unless map_mode 1 with play_min, R36); gen_features reads it for Table
                                IV's "known padded border" (0 = not recorded = the full board) */
    uint32_t *stack_cache;   /* state [N][P+1]  largest owned stack per player + validity stamp, may be NULL (see below) */
    uint32_t *invalid_actions; /* accum [N]  diagnostic, may be NULL: actions since gen_reset that were no pass (R22: k != 0
                                or an index outside [0, 9 H W)) and were not applied -- not the mover's cell, army < 2,
                                target a mountain or off the board, also when an earlier mover of the same turn made
                                them so (R7).  Invalid actions are not errors: they are passes (R5, R10) */
} gen_buffers;

/* `stack_cache` serves the biased policy (gen_policy.bias_thr, R25: "70 % of moves from the largest owned stack"):
 * the per-step kernel's observation pass holds every army value in registers anyway, so it leaves each player's
 * largest owned stack of the state it emits -- ((army + 1) << 10 | (1023 - cell)), ties to the lowest cell, 0 = owns
 * nothing -- in [g][p] and the global step at which that state will be sampled in [g][P]; the next gen_step's
 * sampler takes it from there instead of scanning the army plane.  Derived state like `bitboards`: the sampler reads
 * it only when the handle's previous launch was such a step on this buffer, one global step ago (the handle keeps
 * track; the stamp is a second, per-game check) -- after gen_reset, gen_rollout, gen_observe, a staged-kernel step, a
 * step with explicit actions or gen_set_global_step, and on a fresh handle, it goes back to the scan -- so it is never
 * stale.  Allocate it zeroed.  Results do not depend on it. */

/* `step_epoch` lets consecutive gen_step launches of one handle overlap.  Without it a launch starts working only
 * when the whole previous grid in the stream has completed (griddepcontrol.wait); the batch then moves through the
 * kernel's phases in lock-step and HBM idles while the rules run.  With it, every warp of the register-resident
 * per-step kernel takes a ticket for its group of 4 games when it starts (start[group]++: the number of earlier
 * launches on the group) and records done[group] = ticket + 1 when everything it wrote is visible; a warp begins its
 * work when done[group] equals its ticket instead of waiting for the grid: games are independent, so
 * a launch depends on the previous one only game by game.  Launches then stream through the GPU like the waves of
 * one large launch.  The counters live on the device, so eager launches, CUDA-graph replays and other handles'
 * launches in between need no bookkeeping.  Ordering against everything else is unchanged: kernels that are not
 * gen_step launches never start before a gen_step grid has completed, one warp of every chained grid waits for the
 * previous grid before it exits (grids complete in stream order), and the first gen_step after any other call on the
 * handle (reset, rollout, observe, a staged-kernel step) waits for the whole grid.  A chained launch is therefore
 * ordered on entry ONLY against earlier gen_step launches on the same games of the same buffer set: it consumes
 * nothing else.  A gen_step with explicit `d_actions` (produced by whatever ran before it in the stream: a policy
 * kernel, another handle's gen_step) is never chained -- it waits for its whole stream predecessor before its first
 * global access -- and two handles must not share any buffer.  Allocate it zeroed, once; one handle per buffer
 * set.  Results do not depend on it. */

/* `score_hist` (R34; the paper's two temporal tokens are 512-step windows of
 * the opponent's army and land totals): when non-NULL, gen_reset and every turn of gen_step / gen_rollout store
 * (land[p], army_total[p]) of every player, as the call leaves the scoreboard, in slot (turn mod 512) of the
 * game's ring ([2p] = land, [2p+1] = army).  The last min(turn + 1, 512) slots belong to the current episode;
 * older slots are leftovers.  Frozen games are not recorded. */

/* `obs_packed` (R33) selects the 3-byte-per-cell observation format: when it is non-NULL
 * every call writes obs_army and obs_packed and does NOT write obs_owner / obs_terrain / obs_vis (which may
 * then be NULL).  One byte per cell and player: visible -> 0x80 | terrain << 4 | (owner + 2) (owner + 2: 1 =
 * neutral, 2.. = player 0..); fogged -> 0.  Observation traffic drops from 5 to 3 bytes per cell and player. */

/* `bitboards` caches what the rules need of the three planes as one bit per cell (bit c & 31 of word
 * c >> 5; BW = gen_sizes.bitboard_row_words = ceil(H*W / 32) rounded up to 8 words, so that every row is a whole number of 32-byte sectors): rows 0..P-1 "owned by
 * player p", row P "army >= 2", row P+1 "city or general", row P+2 "mountain or off the board" (all ones
 * past H*W).  gen_reset and gen_observe build it from the planes; gen_step and gen_rollout keep it
 * current.  With it, gen_step without a digest buffer runs the register-resident per-step kernel, which
 * never rebuilds the rows from the planes; without it (NULL) every call stages and scans the planes.
 * A caller who writes the planes directly must call gen_observe before the next gen_step. */

/* byte sizes of the buffers above for K slots */
typedef struct gen_sizes {
    int32_t plane_stride;    /* S in cells */
    int32_t alignment;       /* 16 */
    size_t army, owner, terrain, turn, episode, alive, general_cell, land, army_total;
    size_t reward, done, winner, obs_army, obs_owner, obs_terrain, obs_vis;
    size_t episodes_done, wins, truncations, sat_events, obs_digest, actions_out, bitboards, obs_packed, score_hist;
    size_t step_epoch, play_size, stack_cache, invalid_actions;
    int32_t bitboard_row_words; /* BW */
} gen_sizes;

typedef struct gen_env gen_env;

/* Sizes of every device buffer for `cfg` with `k_slots` >= 1 output slots.  Host-only. */
int gen_query_sizes(const gen_config *cfg, int32_t k_slots, gen_sizes *out);

/* Validate `cfg`, build the host-side handle.  Allocates no device memory.  Policy defaults to
 * pass 0, half 1/2, bias 0.  GEN_ERR_CONFIG on a bad config. */
int gen_init(const gen_config *cfg, gen_env **out);

/* Set the built-in sampler's thresholds (a12; R24, R25). */
int gen_set_policy(gen_env *env, const gen_policy *policy);

/* The spawn-distance curriculum ("we cap the maximum spawn distance ... and gradually raise it over training";
 * P:L118 lists it among the environment's functions): change the spawn window of the boards generated from now on
 * (gen_reset and every auto-reset) without a new handle.  Same meaning and checks as the gen_config fields. */
int gen_set_spawn(gen_env *env, int32_t spawn_dmin, int32_t spawn_dmax, int32_t spawn_exact);

/* Count of steps since gen_reset: the Philox counter word of the action stream. */
uint32_t gen_global_step(const gen_env *env);
int gen_set_global_step(gen_env *env, uint32_t step);

/* a1: generate all N boards (Philox keyed by seed, global game id, episode; R13-R15, R29, R30),
 * zero the accumulators, write scoreboard + initial observation (+ digest if obs_digest != NULL),
 * global_step <- 0.  flags: 0 or GEN_KEEP_EPISODE. */
int gen_reset(gen_env *env, const gen_buffers *bufs, uint32_t flags, void *cuda_stream);

/* a2-a12: one turn for all games.  d_actions: device int32 [N][P] flat action indices
 * a = cell*9 + k, k = 0 pass, else 1 + 2*dir + half, dir 0 up 1 down 2 left 3 right (R22);
 * NULL = draw them with the built-in valid-action sampler.  Writes state, scoreboard, reward, done,
 * winner, the four observation planes per player, actions_out / obs_digest if given.
 * global_step += 1. */
int gen_step(gen_env *env, const gen_buffers *bufs, const int32_t *d_actions, void *cuda_stream);

/* gen_step for callers that cannot allocate device memory.
 *
 * The fast path of gen_step (the register-resident kernel) wants `bufs->bitboards`: working memory that is neither
 * input nor result, which a caller normally allocates once.  Not every caller can.  If your code runs as an operator
 * inside another system's executor (a custom call of a compiled graph, a runtime plug-in) you are given operands and
 * results and no workspace, and you must not call the CUDA allocator yourself; if the learner took all of HBM at
 * start-up, a later cudaMalloc fails; and in an actor loop that must not stall, cudaMalloc / cudaFree are off the
 * table because they synchronise the whole device.  This call is for those cases: it plays one turn exactly like
 * gen_step (same arguments, same outputs, same global_step += 1, bit-identical results) and takes the cache from a
 * fixed array inside the library instead -- GEN_NOALLOC_SCRATCH_BYTES of device memory that every GPU holds from the
 * moment the library is loaded on it until the process ends.  It calls no cudaMalloc, no cudaFree and no library
 * routine that allocates.
 *   - You still pass every input and output in `bufs`.  `bufs->bitboards`, `step_epoch` and `stack_cache` are ignored
 *     (leave them NULL); `bufs->obs_digest` must be NULL and n_players <= 4 (GEN_ERR_ARG otherwise: those steps run
 *     the staged kernel, which needs no cache -- plain gen_step with bitboards = NULL already allocates nothing).
 *   - Limit: n_games * (n_players + 3) * bitboard_row_words * 4 bytes must fit the array, i.e. 17,476 games of 24x24
 *     1v1, 6,553 of 32x32 2v2.  A larger batch is refused with GEN_ERR_SIZE before anything is launched; split it
 *     into several handles (game_id_base) and call them one after the other on one stream.
 *   - The array is shared by every handle and every call in the process and keeps whatever the last call left in it.
 *     That is harmless by construction: each call first rewrites, from your planes, every word the step will read
 *     (one extra small kernel, about 4 bytes read per cell), so nothing has to be cleared and nothing stale is ever
 *     used.  But two calls that run on the GPU AT THE SAME TIME (different streams, different threads, different
 *     handles) write the same array and corrupt each other: keep all gen_step_noalloc calls of a process on one
 *     stream, or order them with events.
 *   - The first call on each device looks up the array's device address (cudaGetSymbolAddress, with that device
 *     current -- so call it with the device you will run on selected).  Make that first call during start-up, before
 *     any stream capture begins.  Later calls on the device only read the remembered address.
 *   - Launches are never chained (each waits for its stream predecessor) and the build pass costs extra traffic, so
 *     callers who CAN allocate should keep using gen_step with their own buffers: this is the slower of the two.
 * Errors as gen_step, plus GEN_ERR_SIZE and GEN_ERR_ARG above; GEN_ERR_CUDA if the address look-up or a launch fails. */
#define GEN_NOALLOC_SCRATCH_BYTES (8u << 20)
int gen_step_noalloc(gen_env *env, const gen_buffers *bufs, const int32_t *d_actions, void *cuda_stream);

/* a13: K sampled turns in ONE launch, the board resident in shared memory throughout (R28).
 * flags: one of GEN_OBS_DIGEST / GEN_OBS_EVERY_STEP / GEN_OBS_NONE.  EVERY_STEP needs buffers sized
 * for K slots.  Otherwise reward / done / winner / planes of the last step land in slot 0.
 * global_step += K. */
int gen_rollout(gen_env *env, const gen_buffers *bufs, int32_t K, uint32_t flags, void *cuda_stream);

/* Recount the scoreboard of a state written by the caller and emit its observation (no turn is
 * played).  For hand-built boards. */
int gen_observe(gen_env *env, const gen_buffers *bufs, void *cuda_stream);

/* The sampler alone (a12): d_actions_out int32 [N][P] drawn on the boards as they stand with the
 * current global_step; no state change. */
int gen_sample(gen_env *env, const gen_buffers *bufs, int32_t *d_actions_out, void *cuda_stream);

/* End-to-end convenience: HOST actions in (int32 [N][P], may be NULL = sampler), HOST results out
 * (reward int8 [N][P], done uint8 [N]; either may be NULL); runs gen_step on cuda_stream and synchronises that stream
 * before returning.  Pinned (page-locked or registered) host buffers are used in place: the step kernel reads the
 * actions through their device alias and writes every game's reward + done to the host arrays as it writes them to
 * the device buffers (posted writes through the mapped aliases; a second small kernel does it where the staged kernel
 * serves the step) -- no copy-engine transfers.  h_actions must have been written by the HOST: a step whose actions
 * sit in pinned host memory chains behind the previous step like one without actions (nothing on the device produced
 * them).  Pageable buffers go through cudaMemcpyAsync (actions via bufs->actions_out, which must
 * then be non-NULL; it must be non-NULL whenever h_actions is given).  Whether a buffer is pinned is looked up when
 * a pinned pointer is passed for the first time (the handle remembers the last eight action arrays and the last eight
 * result arrays; pageable pointers are looked up every call); after unregistering or freeing a pinned buffer call
 * gen_forget_host_buffers. */
int gen_step_host(gen_env *env, const gen_buffers *bufs, const int32_t *h_actions, int8_t *h_reward,
                  uint8_t *h_done, void *cuda_stream);

/* The same without the synchronisation: enqueues the step (and the transfer of reward + done) and returns.  The
 * results of the call issued `lag` calls before the latest one are in their host arrays once gen_host_wait(env, lag)
 * has returned (lag 0 = the latest call; at most 4 calls may be in flight, lag <= 3: a fifth call first waits, inside
 * gen_step_host_async, for the oldest one nobody has waited for).  An RL loop waits one step
 * late -- issue step t with one pair of host slots, then wait for step t - 1 and read the other pair -- so that the
 * GPU always has the next step queued and no launch latency or host wake-up sits between two steps.  Until its wait
 * has returned a call OWNS its three host arrays: pinned actions are read in place when the kernel runs, so they
 * must not be rewritten before.  Use pinned memory: with pageable buffers the copies are staged by the runtime and
 * the call is asynchronous only in name.  The observation planes stay on the device in both variants (a GPU-resident
 * learner reads them there; 94 MB per step at config 2 is no bus traffic to plan for). */
int gen_step_host_async(gen_env *env, const gen_buffers *bufs, const int32_t *h_actions, int8_t *h_reward,
                        uint8_t *h_done, void *cuda_stream);
int gen_host_wait(gen_env *env, int32_t lag);

/* Forget what gen_step_host[_async] has learnt about the caller's host pointers (pinned or not, and their device
 * aliases).  Call it after freeing or unregistering a host buffer that was passed before, so that its address, if
 * the allocator hands it out again, is looked up afresh. */
int gen_forget_host_buffers(gen_env *env);

/* ---- the 38-channel feature tensor (Appendix A, Table IV; R35) ----
 * What the paper's policy consumes, built from the state the step leaves behind plus a per-episode memory.
 * Table IV speaks of "the agent" and "the opponent"; with more than two players (the same observation
 * interface in 1v1, 2v2 and free-for-all; R38) the opponent is every player off the agent's team, visibility is the
 * team's and channels 18 / 19 sum the enemies' scoreboard entries.  Channels, per player p as the agent, float32:
 *   0 armies (visible)  1 own_army  2 enemy_army (visible)  3 neutral_army (visible)
 *   4 seen  5 enemy_seen  6 generals  7 castles  8 mountains          (memory: ever observed, this episode)
 *   9 neutral_cells (visible)  10 owned_cells  11 opponent_cells (visible)  12 fog_cells
 *   13 structures_in_fog (fogged now, remembered general / castle / mountain)
 *   14 timestep (raw turn)  15 (turn mod 50) / 50  16 own land  17 own army  18 opponent land  19 opponent army
 *   20 last_enemy_army_seen  21 log(1 + turns since that sighting) / 5, 0 if never seen or visible now
 *   22 col / (W - 1)  23 row / (H - 1)
 *   24..30 own_army_delta[k], 31..37 enemy_army_delta[k]: frame(t-k) - frame(t-k-1) of channel 1 / 2, k = 0..6,
 *          0 where t-k-1 lies before the episode's first turn.
 * All members are DEVICE pointers, 16-byte aligned, caller-owned; sizes from gen_query_feat_sizes.  The memory
 * members are opaque to the caller: allocate them ZEROED once (a zeroed memory is an empty one) and pass the same
 * ones to every call. */
typedef struct gen_feat_buffers {
    float *feat;         /* out   [N][P][38][S]; stride padding cells are 0 */
    uint8_t *mem_bits;   /* state [N][P][S]     bit k = channel 4 + k */
    int16_t *last_army;  /* state [N][P][S]     channel 20 */
    int32_t *last_seen;  /* state [N][P][S]     turn of the last enemy sighting + 1, 0 = never */
    int16_t *hist;       /* state [N][P][8][2][S]  own_army / enemy_army frames, slot = turn mod 8 */
    uint16_t *feat_bf16; /* out   [N][P][38][S] bfloat16 bit patterns (R37); when non-NULL it is written INSTEAD of
                            feat (which may then be NULL): every fp32 value rounded once, ties to even */
} gen_feat_buffers;

typedef struct gen_feat_sizes {
    int32_t channels;     /* 38 */
    int32_t plane_stride; /* S */
    size_t feat, mem_bits, last_army, last_seen, hist, feat_bf16; /* bytes */
    size_t hist_windows;  /* bytes of gen_history_windows' output: int32 [N][P][2][512] */
} gen_feat_sizes;

/* Byte sizes of the gen_feat_buffers members for `cfg`.  Host-only. */
int gen_query_feat_sizes(const gen_config *cfg, gen_feat_sizes *out);

/* Fold the state as it stands (after gen_reset, gen_step or gen_rollout) into each player's memory and write the
 * feature tensor.  Call it ONCE PER TURN: the delta channels difference consecutive calls' frames, and a game whose
 * turn counter is 0 (fresh or auto-reset, R17) starts from an empty memory.  Reads bufs->army / owner / terrain /
 * turn / land / army_total (and play_size if given) only; no game state changes.  One kernel launch on cuda_stream.
 * GEN_ERR_NULL / GEN_ERR_ALIGN on a missing / misaligned pointer. */
int gen_features(gen_env *env, const gen_buffers *bufs, const gen_feat_buffers *feat, void *cuda_stream);

/* The two temporal tokens' windows ("a 512-step sliding window of the opponent's total army count and a
 * matching window of their total land count, each projected by an MLP into a single token"; reading R39 of
 * DESIGN.md).  Reads bufs->score_hist (the ring of R34, required) and bufs->turn; writes d_windows, caller-owned
 * device memory, int32 [N][P][2][512], 16-byte aligned (gen_feat_sizes.hist_windows bytes): for game g and agent p,
 * [g][p][0][i] is the summed army total and [g][p][1][i] the summed land count of every player off p's team (R38;
 * with two players: the opponent) at turn t - 511 + i of the CURRENT episode, t = turn[g] -- oldest first, entry 511
 * is the scoreboard as it stands now -- and 0 for the entries before the episode's first turn (also the leftovers of an
 * earlier episode in the ring are masked).  The MLP that turns a window into a token is the policy's.  One kernel
 * launch on cuda_stream, no state changes.  GEN_ERR_NULL when the ring was not given, GEN_ERR_ALIGN on a misaligned
 * pointer. */
int gen_history_windows(gen_env *env, const gen_buffers *bufs, int32_t *d_windows, void *cuda_stream);

/* Launch geometry override for tuning: games per CTA in {4, 8, 16, 32} (8 threads per game); 0 restores
 * the default (8).  Results do not depend on it. */
int gen_set_launch(gen_env *env, int32_t games_per_cta);

/* Kernel selection overrides for tests.  The library holds two kernels: the STAGED one (planes resident in
 * shared memory; serves every call) and the REGISTER-RESIDENT per-step one (gen_step with bufs->bitboards
 * and without a digest buffer), each as a generic instantiation for every board up to
 * 32x32 and as instantiations compiled for the paper-sized configurations (1v1 8x8 and 24x24, 4 and 8
 * players on 32x32).  force_generic != 0: never launch a board-specialised instantiation;
 * force_staged == 1: never launch the register-resident kernel; force_staged == -1: launch it
 * whenever it can serve the call (by default games with more than 4 players stay on the staged kernel, which
 * is faster for them).  Results do not depend on either. */
int gen_set_generic(gen_env *env, int32_t force_generic, int32_t force_staged);

/* Launch chaining through gen_buffers.step_epoch (see there): enabled != 0 (default) / 0 = every gen_step waits for
 * the whole previous grid even when step_epoch is given.  Results do not depend on it. */
int gen_set_chaining(gen_env *env, int32_t enabled);

/* Which instantiation the last launch of this handle used: returns its index in the library's variant
 * table (-1 before the first launch); if non-NULL, *board_specialised is set to 1 when that kernel was
 * compiled for this exact board size, *register_resident to 1 when it was the register-resident per-step
 * kernel.  Diagnostic only. */
int32_t gen_last_variant(const gen_env *env, int32_t *board_specialised, int32_t *register_resident);

/* Number of kernels this handle has launched (bench.py's gpu_launches). */
uint64_t gen_launch_count(const gen_env *env);

/* cudaError_t of the last failing runtime call made through this handle (0 if none). */
int gen_last_cuda_error(const gen_env *env);

void gen_destroy(gen_env *env);
const char *gen_error_string(int code);
const char *gen_version(void);

#ifdef __cplusplus
}
#endif
#endif /* GENERALS_H_ */
