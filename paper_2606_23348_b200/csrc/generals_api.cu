// generals_api.cu -- the C ABI of include/generals.h: host-side validation, launch geometry, launches.
// No torch types, no allocation of board memory, no synchronisation (except gen_step_host).
#include <cstdio>
#include <cstring>
#include <new>

#include "generals_variants.h"
#include "generals_features.h"

struct gen_env {
    gen_config cfg;
    gen_policy policy;
    gen::KParams base;       // config-derived fields, filled once
    uint32_t global_step;
    int32_t games_per_cta;   // 0 = default
    uint64_t launches;
    int last_cuda_error;
    int32_t force_generic;   // 1: never pick a board-specialised kernel (tests)
    int32_t force_staged;    // 1: never pick the register-resident step kernel (tests)
    int32_t force_step;      // 1: pick it whenever it can serve the call, also where the staged one is faster (tests)
    int32_t last_variant;    // index into GEN_VARIANTS of the last launch (-1: none yet)
    const uint32_t *chain_buf;  // non-NULL: the last launch of this handle was a k_step that kept records there
    int32_t no_chain;        // tests: never chain
    // non-NULL: the last launch of this handle was a BIAS k_step that left every player's largest stack there, for the
    // state that will be sampled at global step stack_step.  Any other launch, gen_set_global_step or a failed launch
    // clears it: the device-side stamp alone can match again after gen_reset or gen_set_global_step.
    const uint32_t *stack_buf;
    uint32_t stack_step;
    // gen_step_host / gen_step_host_async: host pointers looked up so far and their device aliases (nullptr:
    // pageable memory); a small table, so that double-buffered host slots do not look up again every call
    // Two tables of eight: [0] action arrays (a caller may pass a new one every step), [1] result arrays -- so that a
    // stream of action pointers never evicts the reward / done entries.  Only pinned buffers are remembered: a
    // pageable one is looked up again each call (it may have been registered since).
    const void *hp_key[2][8];
    void *hp_dev[2][8];
    int32_t hp_used[2], hp_next[2];
    // gen_step_host_async: one event per call in flight (ring), created on first use
    cudaEvent_t ev[4];
    int32_t ev_ready;        // events created
    uint64_t async_calls;    // gen_step_host_async calls so far
    uint64_t async_waited;   // the first async_waited of them are known to have completed (gen_host_wait)
    // set by step_host_enqueue around its gen_step call: where k_step also writes reward / done (NULL: nowhere), and
    // whether the actions it passes were written by the HOST (pinned memory read in place: nothing on the device
    // produced them, so the launch may chain)
    int8_t *mirror_reward;
    uint8_t *mirror_done;
    int32_t mirror_armed, mirror_done_in_kernel, actions_from_host;
};

namespace {

inline int round_up(int x, int m) { return (x + m - 1) / m * m; }

int validate(const gen_config *c) {
    if (c->n_games < 0) return GEN_ERR_CONFIG;
    if (c->height < 1 || c->height > 32 || c->width < 1 || c->width > 32) return GEN_ERR_CONFIG;
    if (c->n_players < 2 || c->n_players > 8) return GEN_ERR_CONFIG;
    if (c->height * c->width < c->n_players) return GEN_ERR_CONFIG;
    if (c->team_size < 1 || c->team_size > c->n_players) return GEN_ERR_CONFIG;
    if (c->n_cities < 0 || c->n_cities > c->height * c->width) return GEN_ERR_CONFIG;
    if (c->city_army_lo < 0 || c->city_army_hi < c->city_army_lo || c->city_army_hi > 32767) return GEN_ERR_CONFIG;
    if (c->spawn_dmin < 0 || c->spawn_dmax < 0) return GEN_ERR_CONFIG;
    if (c->spawn_dmax > 0 && c->spawn_dmax < c->spawn_dmin) return GEN_ERR_CONFIG;
    if (c->spawn_exact && c->spawn_dmax <= 0) return GEN_ERR_CONFIG;
    if (c->max_turns < 0) return GEN_ERR_CONFIG;
    if (c->rule_flags & ~7u) return GEN_ERR_CONFIG;
    if ((uint64_t)c->game_id_base + (uint64_t)c->n_games > 0x100000000ull) return GEN_ERR_CONFIG;
    if (c->map_mode != 0 && c->map_mode != 1) return GEN_ERR_CONFIG;
    if (c->map_mode == 0 && (c->n_cities_max || c->play_min || c->castle_radius)) return GEN_ERR_CONFIG;
    if (c->map_mode == 1) {                                    // the official generator (R36): 1v1
        if (c->n_players != 2 || c->team_size != 1) return GEN_ERR_CONFIG;
        if (c->n_cities_max != 0 && c->n_cities_max < c->n_cities) return GEN_ERR_CONFIG;
        if (c->n_cities_max > c->height * c->width) return GEN_ERR_CONFIG;
        if (c->play_min < 0 || c->castle_radius < 0) return GEN_ERR_CONFIG;
        const int hmin = c->play_min > 0 && c->play_min < c->height ? c->play_min : c->height;
        const int wmin = c->play_min > 0 && c->play_min < c->width ? c->play_min : c->width;
        if (hmin * wmin < 2) return GEN_ERR_CONFIG;            // two generals need two cells
    }
    return GEN_OK;
}

void fill_sizes(const gen_config *c, int32_t K, gen_sizes *s) {
    const size_t N = (size_t)c->n_games, P = (size_t)c->n_players, k = (size_t)K;
    const size_t S = (size_t)round_up(c->height * c->width, 16);
    std::memset(s, 0, sizeof(*s));
    s->plane_stride = (int32_t)S;
    s->alignment = 16;
    s->army = N * S * 2; s->owner = N * S; s->terrain = N * S;
    s->turn = N * 4; s->episode = N * 4; s->alive = N; s->general_cell = N * P * 2;
    s->land = N * P * 4; s->army_total = N * P * 4;
    s->reward = k * N * P; s->done = k * N; s->winner = k * N;
    s->obs_army = k * N * P * S * 2; s->obs_owner = k * N * P * S; s->obs_terrain = k * N * P * S;
    s->obs_vis = k * N * P * S;
    s->episodes_done = N * 4; s->wins = N * P * 4; s->truncations = N * 4; s->sat_events = N * 4;
    s->obs_digest = N * 8; s->actions_out = k * N * P * 4;
    const size_t BW = (size_t)round_up((c->height * c->width + 31) / 32, 8);
    s->bitboard_row_words = (int32_t)BW;
    s->bitboards = N * (P + 3) * BW * 4;
    s->obs_packed = k * N * P * S;
    s->score_hist = N * 512 * 2 * P * 4;
    s->step_epoch = (N + 3) / 4 * 8;
    s->play_size = N * 2;
    s->stack_cache = N * (P + 1) * 4;
    s->invalid_actions = N * 4;
}

bool aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

int check_buffers(const gen_buffers *b, bool need_obs) {
    const void *req[] = {b->army, b->owner, b->terrain, b->turn, b->episode, b->alive, b->general_cell,
                         b->land, b->army_total, b->reward, b->done, b->winner, b->episodes_done, b->wins,
                         b->truncations, b->sat_events};
    for (const void *p : req) {
        if (!p) return GEN_ERR_NULL;
        if (!aligned16(p)) return GEN_ERR_ALIGN;
    }
    // observation: army plus either the packed byte plane (R33) or the three byte planes
    const void *obs[] = {b->obs_army, b->obs_owner, b->obs_terrain, b->obs_vis, b->obs_packed};
    for (int i = 0; i < 5; ++i) {
        const bool needed = need_obs && (i == 0 || (b->obs_packed ? i == 4 : i < 4));
        if (needed && !obs[i]) return GEN_ERR_NULL;
        if (obs[i] && !aligned16(obs[i])) return GEN_ERR_ALIGN;
    }
    if (b->obs_digest && !aligned16(b->obs_digest)) return GEN_ERR_ALIGN;
    if (b->actions_out && !aligned16(b->actions_out)) return GEN_ERR_ALIGN;
    if (b->bitboards && !aligned16(b->bitboards)) return GEN_ERR_ALIGN;
    if (b->score_hist && !aligned16(b->score_hist)) return GEN_ERR_ALIGN;
    if (b->step_epoch && !aligned16(b->step_epoch)) return GEN_ERR_ALIGN;
    if (b->play_size && !aligned16(b->play_size)) return GEN_ERR_ALIGN;
    if (b->stack_cache && !aligned16(b->stack_cache)) return GEN_ERR_ALIGN;
    if (b->invalid_actions && !aligned16(b->invalid_actions)) return GEN_ERR_ALIGN;
    return GEN_OK;
}

using gen::kMaxSmem;

inline uint32_t align_up(uint32_t x, uint32_t a) { return (x + a - 1) / a * a; }

// shared-memory layout of one CTA of WPC warps (see generals_kernels.cuh):
// [column / in-bounds tables | digest keys | warp 0 slice | warp 1 slice | ...]
void layout(gen::KParams &k, int WPC, bool digest) {
    k.WPC = WPC;
    const uint32_t GW = (uint32_t)gen::GW, S = (uint32_t)k.S;
    k.off_key = 416;  // three tables of 34 words (zero guards at both ends), 16-byte aligned
    (void)digest;     // the digest keys are a global table (generals_kernels.cuh), no shared memory
    k.off_warp0 = align_up(k.off_key, 128);
    uint32_t off = 2 * GW * S;
    k.w_owner = off; off += GW * S;
    k.w_terr = off; off += GW * S;
    k.w_mask = off; off += GW * (uint32_t)k.M * (uint32_t)k.RW * 4u;
    off = align_up(off, 8);
    k.w_game = off; off += GW * (uint32_t)sizeof(gen::GameS);
    off = align_up(off, 8);
    k.w_bar = off; off += 8;
    k.warp_bytes = align_up(off, 128);
    k.smem_bytes = k.off_warp0 + (uint32_t)WPC * k.warp_bytes;
}

// shared-memory layout of one CTA of the register-resident step kernel (generals_step.cuh):
// [tables | warp 0: cache rows, vis rows, scalars, mbarrier, regeneration scratch | warp 1 | ...]
void layout_step(gen::KParams &k, int WPC) {
    k.WPC = WPC;
    const uint32_t GW = (uint32_t)gen::GW, P = (uint32_t)k.P, BW = (uint32_t)k.BW;
    k.off_key = 416;
    k.off_warp0 = 512;
    uint32_t off = GW * (2 * P + 3) * BW * 4u;
    k.w_mask = 0;
    k.w_game = off; off += GW * (uint32_t)sizeof(gen::StepGame);
    k.w_bar = off; off += 8;
    off = align_up(off, 16);
    k.w_scratch = off; off += 4u * (uint32_t)k.S;
    k.warp_bytes = align_up(off, 128);
    k.smem_bytes = k.off_warp0 + (uint32_t)WPC * k.warp_bytes;
}

constexpr long kSMs = 148;  // B200
using gen::F_RUNTIME;
using gen::F_OBS_PLANES;
using gen::F_OBS_EVERY;
using gen::F_RESET;
using gen::FF_ROLL_DIGEST;
const gen::Variant kVariants[gen::N_VARIANTS] = {
#define GEN_ROW(id, kind, np, h, w, ff, maxt, minb) {kind, np, h, w, ff, maxt, minb, gen::launch_variant_##id},
    GEN_VARIANTS(GEN_ROW)
#undef GEN_ROW
};

// The most specialised instantiation that serves this launch.  step_ok: the register-resident kernel may
// be used (gen_step with the bitboard cache, no digest).  Within a kind: the exact board
// (and, for the staged kernel, the exact mode) first, else the generic kernel of the smallest NP >= P.
const gen::Variant *pick_variant(const gen_env *env, const gen::KParams &kp, bool step_ok) {
    const int kind = (step_ok ? 1 : 0) + (kp.map_mode == 1 ? 2 : 0);
    const gen::Variant *generic = nullptr, *exact = nullptr;
    // k_step: ff = 1 is the build whose observation pass also finds each player's largest stack (stack_cache) for
    // the biased policy; where the board has no such build the plain one serves (its sampler scans the army plane)
    const bool want_stack = (kind & 1) && kp.bias_thr != 0 && (kp.flags & gen::F_SAMPLER) && kp.b.stack_cache != nullptr;
    for (int pass = want_stack ? 0 : 1; pass < 2 && !exact; ++pass)
    for (const gen::Variant &v : kVariants) {
        if (v.kind != kind) continue;
        if (v.h == 0) {
            if (kp.P <= v.np && (!generic || v.np < generic->np)) generic = &v;
            continue;
        }
        if (env->force_generic || v.np != kp.P || v.h != kp.H || v.w != kp.W) continue;
        if (v.np == 2 && kp.team_size > 1) continue;
        if ((kind & 1) == 0 && v.ff != (kp.flags & ~gen::F_SAMPLER)) continue;
        if ((kind & 1) == 1 && (v.ff != 0) != (pass == 0)) continue;
        if (!exact) { exact = &v; continue; }
        // the same kernel under several register budgets (resident CTAs per SM): 12 for batches below one wave of it,
        // 14 up to the size where launches stop chaining (launch()) -- only that holds config 2's batch resident in
        // one wave --, else 10; the closest budget on offer wins, the roomier one on a tie
        const long ctas = (kp.N + 2 * gen::GW - 1) / (2 * gen::GW);
        // (round 2, rotation of replicas, 72- against 80-register build: equal at 24,576 and 32,768 games, 97.2 against
        // 98.5 us at 65,536, 194.3 against 197.0 us at 131,072 -- so 14 wherever the launches still chain)
        // (beyond that size: four planes 391 us at 10 against 406 us at 14 CTAs per SM for 262,144 games; the packed
        // observation, with 40 % fewer bytes to store per step, 325 us at 10 against 305 us at 14)
        const int want = ctas <= 12 * kSMs ? 12 : (ctas <= 8 * 14 * kSMs || kp.b.obs_packed) ? 14 : 10;
        const int dv = v.min_ctas > want ? v.min_ctas - want : want - v.min_ctas;
        const int de = exact->min_ctas > want ? exact->min_ctas - want : want - exact->min_ctas;
        if (dv < de || (dv == de && v.min_ctas < exact->min_ctas)) exact = &v;
    }
    if (exact) return exact;
    return generic;
}

int launch(gen_env *env, const gen_buffers *bufs, uint32_t flags, int32_t K, const int32_t *actions,
           int32_t *sample_out, void *stream) {
    if (env->cfg.n_games == 0) return GEN_OK;
    gen::KParams kp = env->base;
    kp.pass_thr = env->policy.pass_thr;
    kp.half_thr = env->policy.half_thr;
    kp.bias_thr = env->policy.bias_thr;
    kp.global_step0 = env->global_step;
    kp.flags = flags;
    kp.K = K;
    kp.b = *bufs;
    kp.actions = actions;
    kp.sample_out = sample_out;
    // gen_step proper (one turn, planes, no digest) with the bitboard cache runs the register-resident kernel;
    // everything else the staged one
    // (more than 4 players: one lane per player in the word passes and 8 x 4 half-written lines per chunk in the
    // emit pass -- measured 2x the DRAM traffic and half the speed of the staged kernel, so those stay there)
    const bool step_ok = !env->force_staged && K == 1 && bufs->bitboards &&
                         (flags & ~gen::F_SAMPLER) == gen::F_OBS_PLANES && (kp.P <= 4 || env->force_step);
    const gen::Variant *v = pick_variant(env, kp, step_ok);
    if (!v) return GEN_ERR_CONFIG;
    // warps per CTA (4 games each): 2 by default; fewer while the CTA would not fit
    int WPC = env->games_per_cta ? env->games_per_cta / gen::GW : 2;
    while (32 * WPC > v->max_threads) WPC >>= 1;
    const bool digest = (flags & gen::F_DIGEST) != 0;
    if (v->kind & 1) layout_step(kp, WPC); else layout(kp, WPC, digest);
    // staged kernel, default geometry: big boards with many players are limited by shared memory (7.4 KB per game at
    // 32x32 with 8 players); one warp per CTA then packs more games onto an SM (FFA-8: 28 instead of 24, +9 %)
    if (!(v->kind & 1) && !env->games_per_cta && WPC == 2) {
        auto resident = [&](int w) {
            layout(kp, w, digest);
            const long ctas = 232448L / ((long)kp.smem_bytes + 1024L);
            return (ctas < 32 ? ctas : 32) * gen::GW * w;
        };
        const long r2 = resident(2), r1 = resident(1);
        if (r1 > r2) WPC = 1;
        layout(kp, WPC, digest);
    }
    while (WPC > 1 && kp.smem_bytes > kMaxSmem) {
        WPC >>= 1;
        if (v->kind & 1) layout_step(kp, WPC); else layout(kp, WPC, digest);
    }
    if (kp.smem_bytes > kMaxSmem) return GEN_ERR_CONFIG;
    const int per_cta = gen::GW * kp.WPC;
    const int grid = (kp.N + per_cta - 1) / per_cta;
    // launch chaining (gen_buffers.step_epoch): a k_step launch waits warp by warp for the earlier k_step launches on
    // the same games instead of for the whole previous grid -- unless the previous call on this handle was something
    // else (a staged-kernel launch triggers its dependents early too and keeps no records)
    // (measured on config 2's boards: chained launches sustain 290 / 490 / 620-660 M env steps/s at 2,048 / 4,096 /
    // 8,192-131,072 games against 118 / 227 / 420-653 M with the grid-wide wait; beyond ~8 waves the waves of one
    // launch mix the phases by themselves and the record's release costs 1-2 %, so those launches keep no records)
    kp.mirror_reward = nullptr; kp.mirror_done = nullptr;
    env->mirror_done_in_kernel = 0;
    if ((v->kind & 1) && env->mirror_armed) {
        kp.mirror_reward = env->mirror_reward; kp.mirror_done = env->mirror_done;
        env->mirror_done_in_kernel = 1;
    }
    kp.count = ((v->kind & 1) && bufs->step_epoch && !env->no_chain && grid <= 8 * 14 * (int)kSMs) ? 1 : 0;
    // A chained launch skips the grid-wide wait, so it may consume nothing a foreign kernel produced: with explicit
    // actions (written by whatever ran before this call) the launch always waits for its stream predecessor.
    kp.chain = (kp.count && env->chain_buf == bufs->step_epoch && (!actions || env->actions_from_host)) ? 1 : 0;
    // gen_buffers.stack_cache is trusted only when the previous launch of this handle was the BIAS build of k_step on
    // the same buffer, one global step ago (like chain_buf: validity is the host's knowledge, the stamp a second check)
    const bool bias_build = (v->kind & 1) && v->ff != 0;
    kp.stack_ok = (bias_build && env->stack_buf && env->stack_buf == bufs->stack_cache &&
                   env->stack_step == env->global_step) ? 1 : 0;
    cudaError_t e = v->launch(kp, grid, 32 * kp.WPC, kp.smem_bytes, static_cast<cudaStream_t>(stream));
    if (e != cudaSuccess) {
        env->last_cuda_error = (int)e; env->chain_buf = nullptr; env->stack_buf = nullptr;
        return GEN_ERR_CUDA;
    }
    env->chain_buf = kp.count ? bufs->step_epoch : nullptr;
    env->stack_buf = bias_build ? bufs->stack_cache : nullptr;
    env->stack_step = env->global_step + 1u;
    env->launches += 1;
    env->last_variant = (int32_t)(v - kVariants);
    return GEN_OK;
}

// gen_step_host with pinned host buffers: one kernel carries reward [N][P] and done [N] to the mapped host memory
// (two byte ranges, 16-byte vectors where the alignment allows) instead of two copy-engine transfers.
__global__ void k_mirror(const unsigned char *__restrict__ src0, unsigned char *__restrict__ dst0, size_t n0,
                         const unsigned char *__restrict__ src1, unsigned char *__restrict__ dst1, size_t n1) {
    const size_t tid = (size_t)blockIdx.x * blockDim.x + threadIdx.x, nthr = (size_t)gridDim.x * blockDim.x;
    for (int r = 0; r < 2; ++r) {
        const unsigned char *src = r ? src1 : src0;
        unsigned char *dst = r ? dst1 : dst0;
        const size_t n = r ? n1 : n0;
        if (!dst || !n) continue;
        if ((((uintptr_t)src | (uintptr_t)dst) & 15u) == 0) {
            const size_t nv = n / 16;
            for (size_t i = tid; i < nv; i += nthr)
                reinterpret_cast<uint4 *>(dst)[i] = reinterpret_cast<const uint4 *>(src)[i];
            for (size_t i = nv * 16 + tid; i < n; i += nthr) dst[i] = src[i];
        } else {
            for (size_t i = tid; i < n; i += nthr) dst[i] = src[i];
        }
    }
}

// device alias of a host pointer that the GPU can access directly (pinned / registered memory), else nullptr
void *mapped_alias(const void *h) {
    if (!h) return nullptr;
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, h) != cudaSuccess) { (void)cudaGetLastError(); return nullptr; }
    if (at.type != cudaMemoryTypeHost) return nullptr;
    return at.devicePointer;
}

uint64_t host_mix64(uint64_t z) {  // splitmix64 finaliser: the digest keys of R28
    z ^= z >> 30; z *= 0xBF58476D1CE4E5B9ull;
    z ^= z >> 27; z *= 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

}  // namespace

namespace gen {
// for generals_noalloc.cu, to which gen_env is an opaque type: the handle's configuration and its launch counter
const gen_config *env_config(const gen_env *env) { return &env->cfg; }
void env_count_launch(gen_env *env) { env->launches += 1; }
}  // namespace gen

extern "C" {

int gen_query_sizes(const gen_config *cfg, int32_t k_slots, gen_sizes *out) {
    if (!cfg || !out) return GEN_ERR_NULL;
    if (int e = validate(cfg)) return e;
    if (k_slots < 1) return GEN_ERR_ARG;
    fill_sizes(cfg, k_slots, out);
    return GEN_OK;
}

int gen_init(const gen_config *cfg, gen_env **out) {
    if (!cfg || !out) return GEN_ERR_NULL;
    *out = nullptr;
    if (int e = validate(cfg)) return e;
    gen_env *env = new (std::nothrow) gen_env();
    if (!env) return GEN_ERR_ARG;
    std::memset(env, 0, sizeof(*env));
    env->cfg = *cfg;
    env->last_variant = -1;
    env->policy.pass_thr = 0;
    env->policy.half_thr = 0x80000000u;
    env->policy.bias_thr = 0;
    gen::KParams &k = env->base;
    k.N = cfg->n_games; k.H = cfg->height; k.W = cfg->width; k.P = cfg->n_players;
    k.HW = k.H * k.W; k.S = round_up(k.HW, 16); k.NW = (k.HW + 31) / 32; k.NC8 = k.S / 8;
    k.NCH = 4 * k.NW; k.RW = k.NW | 1; k.M = 2 * k.P + 7; k.BW = round_up(k.NW, 8);
    k.team_size = cfg->team_size;
    k.n_teams = (cfg->n_players + cfg->team_size - 1) / cfg->team_size;
    k.n_cities = cfg->n_cities; k.city_lo = cfg->city_army_lo;
    k.city_span = cfg->city_army_hi - cfg->city_army_lo + 1;
    k.dmin = cfg->spawn_dmin; k.dmax = cfg->spawn_dmax; k.spawn_exact = cfg->spawn_exact;
    k.max_turns = cfg->max_turns; k.auto_reset = cfg->auto_reset;
    k.map_mode = cfg->map_mode; k.n_cities_max = cfg->n_cities_max; k.play_min = cfg->play_min;
    k.castle_radius = cfg->castle_radius;
    k.rule_flags = cfg->rule_flags; k.gid_base = cfg->game_id_base; k.mountain_thr = cfg->mountain_thr;
    k.key0 = (uint32_t)(cfg->seed & 0xffffffffu); k.key1 = (uint32_t)(cfg->seed >> 32);
    // row = (cell * recipW) >> 16 must equal cell / W for every cell of the largest board
    k.recipW = 65536u / (uint32_t)k.W + 1u;
    for (uint32_t c = 0; c < 1024u; ++c)
        if (((c * k.recipW) >> 16) != c / (uint32_t)k.W) { delete env; return GEN_ERR_CONFIG; }
    k.key_sum = 0;
    for (int c = 0; c < k.HW; ++c) k.key_sum += host_mix64((uint64_t)(c + 1) * 0x9E3779B97F4A7C15ull) | 1ull;
    for (int j = 0; j < 32; ++j) {
        uint32_t n0 = 0, nl = 0, in = 0;
        for (int b = 0; b < 32; ++b) {
            const int c = 32 * j + b;
            if (c >= k.HW) continue;
            in |= 1u << b;
            if (c % k.W != 0) n0 |= 1u << b;
            if (c % k.W != k.W - 1) nl |= 1u << b;
        }
        k.notcol0[j] = n0; k.notcolL[j] = nl; k.inb[j] = in;
    }
    *out = env;
    return GEN_OK;
}

int gen_set_policy(gen_env *env, const gen_policy *policy) {
    if (!env || !policy) return GEN_ERR_NULL;
    env->policy = *policy;
    return GEN_OK;
}

int gen_set_spawn(gen_env *env, int32_t spawn_dmin, int32_t spawn_dmax, int32_t spawn_exact) {
    if (!env) return GEN_ERR_NULL;
    gen_config c = env->cfg;
    c.spawn_dmin = spawn_dmin; c.spawn_dmax = spawn_dmax; c.spawn_exact = spawn_exact ? 1 : 0;
    if (int e = validate(&c)) return e;
    env->cfg = c;
    env->base.dmin = c.spawn_dmin; env->base.dmax = c.spawn_dmax; env->base.spawn_exact = c.spawn_exact;
    return GEN_OK;
}

uint32_t gen_global_step(const gen_env *env) { return env ? env->global_step : 0u; }

int gen_set_global_step(gen_env *env, uint32_t step) {
    if (!env) return GEN_ERR_NULL;
    env->global_step = step;
    env->stack_buf = nullptr;
    return GEN_OK;
}

int gen_reset(gen_env *env, const gen_buffers *bufs, uint32_t flags, void *cuda_stream) {
    if (!env || !bufs) return GEN_ERR_NULL;
    if (flags & ~(uint32_t)GEN_KEEP_EPISODE) return GEN_ERR_ARG;
    if (int e = check_buffers(bufs, true)) return e;
    env->global_step = 0;
    uint32_t f = gen::F_RESET | gen::F_OBS_PLANES;
    if (flags & GEN_KEEP_EPISODE) f |= gen::F_KEEP_EPISODE;
    if (bufs->obs_digest) f |= gen::F_DIGEST;
    return launch(env, bufs, f, 0, nullptr, nullptr, cuda_stream);
}

int gen_step(gen_env *env, const gen_buffers *bufs, const int32_t *d_actions, void *cuda_stream) {
    if (!env || !bufs) return GEN_ERR_NULL;
    if (int e = check_buffers(bufs, true)) return e;
    if (d_actions && !aligned16(d_actions)) return GEN_ERR_ALIGN;
    uint32_t f = gen::F_OBS_PLANES;
    if (!d_actions) f |= gen::F_SAMPLER;
    if (bufs->obs_digest) f |= gen::F_DIGEST;
    const int e = launch(env, bufs, f, 1, d_actions, nullptr, cuda_stream);
    if (e == GEN_OK) env->global_step += 1;
    return e;
}

int gen_rollout(gen_env *env, const gen_buffers *bufs, int32_t K, uint32_t flags, void *cuda_stream) {
    if (!env || !bufs) return GEN_ERR_NULL;
    if (K <= 0) return GEN_ERR_ARG;
    if (flags != GEN_OBS_DIGEST && flags != GEN_OBS_EVERY_STEP && flags != GEN_OBS_NONE) return GEN_ERR_ARG;
    if (int e = check_buffers(bufs, flags != GEN_OBS_NONE)) return e;
    if (flags == GEN_OBS_DIGEST && !bufs->obs_digest) return GEN_ERR_NULL;
    uint32_t f = gen::F_SAMPLER;
    if (flags == GEN_OBS_DIGEST) f |= gen::F_DIGEST | gen::F_OBS_PLANES;
    if (flags == GEN_OBS_EVERY_STEP) {
        f |= gen::F_OBS_PLANES | gen::F_OBS_EVERY;
        if (bufs->obs_digest) f |= gen::F_DIGEST;
    }
    const int e = launch(env, bufs, f, K, nullptr, nullptr, cuda_stream);
    if (e == GEN_OK) env->global_step += (uint32_t)K;
    return e;
}

int gen_observe(gen_env *env, const gen_buffers *bufs, void *cuda_stream) {
    if (!env || !bufs) return GEN_ERR_NULL;
    if (int e = check_buffers(bufs, true)) return e;
    return launch(env, bufs, gen::F_OBSERVE_ONLY | gen::F_OBS_PLANES, 0, nullptr, nullptr, cuda_stream);
}

int gen_sample(gen_env *env, const gen_buffers *bufs, int32_t *d_actions_out, void *cuda_stream) {
    if (!env || !bufs || !d_actions_out) return GEN_ERR_NULL;
    if (int e = check_buffers(bufs, false)) return e;
    return launch(env, bufs, gen::F_SAMPLE_ONLY | gen::F_SAMPLER, 0, nullptr, d_actions_out, cuda_stream);
}

static void *host_alias(gen_env *env, const void *h, int table) {
    if (!h) return nullptr;
    for (int i = 0; i < env->hp_used[table]; ++i)
        if (env->hp_key[table][i] == h) return env->hp_dev[table][i];
    void *dev = mapped_alias(h);
    if (!dev) return nullptr;                                  // pageable: not remembered
    const int slot = env->hp_used[table] < 8 ? env->hp_used[table]++ : (env->hp_next[table]++ & 7);
    env->hp_key[table][slot] = h;
    env->hp_dev[table][slot] = dev;
    return dev;
}

// the body of gen_step_host / gen_step_host_async: everything but the wait
static int step_host_enqueue(gen_env *env, const gen_buffers *bufs, const int32_t *h_actions, int8_t *h_reward,
                             uint8_t *h_done, cudaStream_t s) {
    if (h_actions && !bufs->actions_out) return GEN_ERR_NULL;
    if (int e = check_buffers(bufs, true)) return e;         // before anything is enqueued
    const size_t N = (size_t)env->cfg.n_games, P = (size_t)env->cfg.n_players;
    cudaError_t ce = cudaSuccess;
    // Pinned host buffers are used in place: the step kernel reads the actions through their device alias and one
    // small kernel writes reward + done into the host arrays (no copy-engine transfers).  Pageable buffers take the
    // cudaMemcpyAsync route.  The alias lookups are cached per handle (same buffers every step in an RL loop).
    void *const a_act = host_alias(env, h_actions, 0), *const a_rew = host_alias(env, h_reward, 1),
                *const a_done = host_alias(env, h_done, 1);
    const int32_t *d_act = nullptr;
    if (h_actions) {
        if (a_act && aligned16(a_act)) {
            d_act = static_cast<const int32_t *>(a_act);
        } else {
            ce = cudaMemcpyAsync(bufs->actions_out, h_actions, N * P * 4, cudaMemcpyHostToDevice, s);
            if (ce != cudaSuccess) { env->last_cuda_error = (int)ce; return GEN_ERR_CUDA; }
            d_act = bufs->actions_out;
        }
    }
    const bool mirror = N > 0 && (!h_reward || a_rew) && (!h_done || a_done) && (h_reward || h_done);
    // the step kernel writes a two-player reward row as one 16-bit store: a pinned array at an odd address (a slice of
    // a byte buffer) is served by k_mirror below, which copies byte by byte when it has to
    const bool rew_ok = !h_reward || P != 2 || (reinterpret_cast<uintptr_t>(a_rew) & 1u) == 0;
    env->mirror_armed = (mirror && rew_ok) ? 1 : 0;
    env->mirror_reward = h_reward ? static_cast<int8_t *>(a_rew) : nullptr;
    env->mirror_done = h_done ? static_cast<uint8_t *>(a_done) : nullptr;
    env->actions_from_host = (d_act && d_act == static_cast<const int32_t *>(a_act)) ? 1 : 0;
    const int e = gen_step(env, bufs, d_act, s);
    env->mirror_armed = 0;
    env->actions_from_host = 0;
    if (e != GEN_OK) return e;
    if (mirror && env->mirror_done_in_kernel) {
        // the step kernel has written reward + done to the host arrays as well: nothing to launch
    } else if (mirror) {
        const size_t bytes = N * P + N;
        const int threads = 256, blocks = (int)((bytes / 16 + threads) / threads < 296 ? (bytes / 16 + threads) / threads : 296);
        // (a plain launch on purpose: as a programmatic dependent launch its CTAs would sit on 13 SMs while the next
        // step's grid is placed, and that grid -- exactly one wave at config 2 -- would no longer fit: measured 425 M
        // against 485 M env steps/s end to end)
        k_mirror<<<blocks, threads, 0, s>>>(reinterpret_cast<const unsigned char *>(bufs->reward),
                                            static_cast<unsigned char *>(a_rew), h_reward ? N * P : 0,
                                            bufs->done, static_cast<unsigned char *>(a_done), h_done ? N : 0);
        ce = cudaGetLastError();
        if (ce == cudaSuccess) env->launches += 1;
    } else {
        if (h_reward) ce = cudaMemcpyAsync(h_reward, bufs->reward, N * P, cudaMemcpyDeviceToHost, s);
        if (ce == cudaSuccess && h_done) ce = cudaMemcpyAsync(h_done, bufs->done, N, cudaMemcpyDeviceToHost, s);
    }
    if (ce != cudaSuccess) { env->last_cuda_error = (int)ce; return GEN_ERR_CUDA; }
    return GEN_OK;
}

int gen_step_host(gen_env *env, const gen_buffers *bufs, const int32_t *h_actions, int8_t *h_reward,
                  uint8_t *h_done, void *cuda_stream) {
    if (!env || !bufs) return GEN_ERR_NULL;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    if (int e = step_host_enqueue(env, bufs, h_actions, h_reward, h_done, s)) return e;
    const cudaError_t ce = cudaStreamSynchronize(s);
    if (ce != cudaSuccess) { env->last_cuda_error = (int)ce; return GEN_ERR_CUDA; }
    return GEN_OK;
}

int gen_step_host_async(gen_env *env, const gen_buffers *bufs, const int32_t *h_actions, int8_t *h_reward,
                        uint8_t *h_done, void *cuda_stream) {
    if (!env || !bufs) return GEN_ERR_NULL;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    if (!env->ev_ready) {
        for (int i = 0; i < 4; ++i) {
            const cudaError_t ce = cudaEventCreateWithFlags(&env->ev[i], cudaEventDisableTiming);
            if (ce != cudaSuccess) {
                for (int j = 0; j < i; ++j) cudaEventDestroy(env->ev[j]);
                env->last_cuda_error = (int)ce;
                return GEN_ERR_CUDA;
            }
        }
        env->ev_ready = 1;
    }
    // at most four calls in flight: the event this call records is the one of the call issued four calls ago -- if
    // nobody has waited for that one yet, wait for it here instead of losing track of it
    if (env->async_calls - env->async_waited >= 4) {
        const cudaError_t we = cudaEventSynchronize(env->ev[env->async_calls & 3]);
        if (we != cudaSuccess) { env->last_cuda_error = (int)we; return GEN_ERR_CUDA; }
        env->async_waited = env->async_calls - 3;
    }
    const uint32_t step_before = env->global_step;
    const int e = step_host_enqueue(env, bufs, h_actions, h_reward, h_done, s);
    if (e != GEN_OK && env->global_step == step_before) return e;   // nothing was launched
    // also when a transfer behind the launched step failed: the step counts as a call, so that gen_host_wait(0) waits
    // for it and not for its predecessor
    const cudaError_t ce = cudaEventRecord(env->ev[env->async_calls & 3], s);
    env->async_calls += 1;
    if (e != GEN_OK) return e;
    if (ce != cudaSuccess) { env->last_cuda_error = (int)ce; return GEN_ERR_CUDA; }
    return GEN_OK;
}

int gen_host_wait(gen_env *env, int32_t lag) {
    if (!env) return GEN_ERR_NULL;
    if (lag < 0 || lag > 3) return GEN_ERR_ARG;
    if (env->async_calls <= (uint64_t)lag) return GEN_OK;     // nothing that old has been issued
    const uint64_t call = env->async_calls - 1 - (uint64_t)lag;
    if (call < env->async_waited) return GEN_OK;               // already known to have completed
    const cudaError_t ce = cudaEventSynchronize(env->ev[call & 3]);
    if (ce != cudaSuccess) { env->last_cuda_error = (int)ce; return GEN_ERR_CUDA; }
    env->async_waited = call + 1;                              // stream order: everything before it has completed too
    return GEN_OK;
}

int gen_forget_host_buffers(gen_env *env) {
    if (!env) return GEN_ERR_NULL;
    env->hp_used[0] = env->hp_used[1] = env->hp_next[0] = env->hp_next[1] = 0;
    return GEN_OK;
}

int gen_query_feat_sizes(const gen_config *cfg, gen_feat_sizes *out) {
    if (!cfg || !out) return GEN_ERR_NULL;
    if (int e = validate(cfg)) return e;
    const size_t N = (size_t)cfg->n_games, S = (size_t)round_up(cfg->height * cfg->width, 16);
    const size_t P = (size_t)cfg->n_players;
    std::memset(out, 0, sizeof(*out));
    out->channels = 38;
    out->plane_stride = (int32_t)S;
    out->feat = N * P * 38 * S * 4;
    out->mem_bits = N * P * S;
    out->last_army = N * P * S * 2;
    out->last_seen = N * P * S * 4;
    out->hist = N * P * 8 * 2 * S * 2;
    out->feat_bf16 = N * P * 38 * S * 2;
    out->hist_windows = N * P * 2 * 512 * 4;
    return GEN_OK;
}

int gen_features(gen_env *env, const gen_buffers *bufs, const gen_feat_buffers *feat, void *cuda_stream) {
    if (!env || !bufs || !feat) return GEN_ERR_NULL;
    const void *out = feat->feat_bf16 ? (const void *)feat->feat_bf16 : (const void *)feat->feat;
    if (feat->feat && !aligned16(feat->feat)) return GEN_ERR_ALIGN;
    const void *req[] = {bufs->army, bufs->owner, bufs->terrain, bufs->turn, bufs->land, bufs->army_total,
                         out, feat->mem_bits, feat->last_army, feat->last_seen, feat->hist};
    for (const void *p : req) {
        if (!p) return GEN_ERR_NULL;
        if (!aligned16(p)) return GEN_ERR_ALIGN;
    }
    if (env->cfg.n_games == 0) return GEN_OK;
    gen::FeatParams fp;
    fp.N = env->base.N; fp.H = env->base.H; fp.W = env->base.W; fp.HW = env->base.HW; fp.S = env->base.S;
    fp.P = env->base.P; fp.team_size = env->base.team_size;
    // 2 * S / 4 threads per game; small boards share a CTA of about 256 threads
    const int per_game = fp.S / 2;
    fp.G = per_game >= 256 ? 1 : 256 / per_game;
    fp.force_generic = env->force_generic;
    fp.army = bufs->army; fp.owner = bufs->owner; fp.terrain = bufs->terrain; fp.turn = bufs->turn;
    fp.land = bufs->land; fp.army_total = bufs->army_total; fp.play_size = bufs->play_size;
    fp.feat = const_cast<void *>(out); fp.bf16 = feat->feat_bf16 ? 1 : 0; fp.mem_bits = feat->mem_bits; fp.last_army = feat->last_army;
    fp.last_seen = feat->last_seen; fp.hist = feat->hist;
    const cudaError_t e = gen::launch_features(fp, static_cast<cudaStream_t>(cuda_stream));
    if (e != cudaSuccess) { env->last_cuda_error = (int)e; return GEN_ERR_CUDA; }
    env->launches += 1;
    return GEN_OK;
}

int gen_history_windows(gen_env *env, const gen_buffers *bufs, int32_t *d_windows, void *cuda_stream) {
    if (!env || !bufs || !d_windows || !bufs->score_hist || !bufs->turn) return GEN_ERR_NULL;
    if (!aligned16(d_windows) || !aligned16(bufs->score_hist) || !aligned16(bufs->turn)) return GEN_ERR_ALIGN;
    if (env->cfg.n_games == 0) return GEN_OK;
    const cudaError_t e = gen::launch_history_windows(bufs->score_hist, bufs->turn, d_windows, env->base.N, env->base.P,
                                                      env->base.team_size, static_cast<cudaStream_t>(cuda_stream));
    if (e != cudaSuccess) { env->last_cuda_error = (int)e; return GEN_ERR_CUDA; }
    env->launches += 1;
    return GEN_OK;
}

int gen_set_launch(gen_env *env, int32_t games_per_cta) {
    if (!env) return GEN_ERR_NULL;
    if (games_per_cta != 0 && games_per_cta != 4 && games_per_cta != 8 && games_per_cta != 16 &&
        games_per_cta != 32)
        return GEN_ERR_ARG;
    env->games_per_cta = games_per_cta;
    return GEN_OK;
}

int gen_set_generic(gen_env *env, int32_t force_generic, int32_t force_staged) {
    if (!env) return GEN_ERR_NULL;
    env->force_generic = force_generic ? 1 : 0;
    env->force_staged = force_staged == 1 ? 1 : 0;
    env->force_step = force_staged == -1 ? 1 : 0;
    return GEN_OK;
}

int gen_set_chaining(gen_env *env, int32_t enabled) {
    if (!env) return GEN_ERR_NULL;
    env->no_chain = enabled ? 0 : 1;
    env->chain_buf = nullptr;
    return GEN_OK;
}

int32_t gen_last_variant(const gen_env *env, int32_t *board_specialised, int32_t *register_resident) {
    if (!env || env->last_variant < 0) return -1;
    if (board_specialised) *board_specialised = kVariants[env->last_variant].h > 0 ? 1 : 0;
    if (register_resident) *register_resident = (kVariants[env->last_variant].kind & 1) ? 1 : 0;
    return env->last_variant;
}

uint64_t gen_launch_count(const gen_env *env) { return env ? env->launches : 0; }
int gen_last_cuda_error(const gen_env *env) { return env ? env->last_cuda_error : 0; }

void gen_destroy(gen_env *env) {
    if (env && env->ev_ready)
        for (int i = 0; i < 4; ++i) cudaEventDestroy(env->ev[i]);
    delete env;
}

const char *gen_error_string(int code) {
    switch (code) {
        case GEN_OK: return "ok";
        case GEN_ERR_NULL: return "a required pointer is NULL";
        case GEN_ERR_CONFIG: return "invalid configuration";
        case GEN_ERR_ALIGN: return "device pointer not 16-byte aligned";
        case GEN_ERR_ARG: return "invalid argument";
        case GEN_ERR_CUDA: return "CUDA runtime error (see gen_last_cuda_error)";
        case GEN_ERR_SIZE: return "batch too large for the built-in scratch of gen_step_noalloc (GEN_NOALLOC_SCRATCH_BYTES)";
        default: return "unknown error code";
    }
}

const char *gen_version(void) { return "generals-b200 0.2 (sm_100a)"; }

}  // extern "C"
